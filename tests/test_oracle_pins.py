"""Pins for oracle/herald_oracle.py: every oracle function is checked against something
other than itself -- closed forms, brute-force pure-Python loops, library routines
(torch SDPA fp64, scipy softmax, torch.index_select), invariants -- chosen so that a
dropped term, a wrong sign/index or a transposed operand fails at least one of them.
All CPU (-m "not gpu")."""
import math
import os

import numpy as np
import pytest
import torch

from oracle import herald_oracle as O
from paper_2606_21633_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def bf16_bits(x):
    """float array -> bf16 bit patterns (round-to-nearest-even via torch)."""
    t = torch.as_tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16)
    return synth.to_u16(t)


def bf16_round(x):
    return O.bf16_bits_to_f64(bf16_bits(x))


# ---------------------------------------------------------------- bf16 widening
def test_bf16_widening_known_patterns():
    # IEEE bf16 = top 16 bits of fp32: 0x3F80 = 1.0, 0xC000 = -2.0, 0x3DCD = 0.10009765625, 0x0000 = 0, 0x7F7F = max
    got = O.bf16_bits_to_f64(np.array([0x3F80, 0xC000, 0x3DCD, 0x0000, 0x7F7F, 0x0080], dtype=np.uint16))
    want = [1.0, -2.0, 0.10009765625, 0.0, (2 - 2 ** -7) * 2.0 ** 127, 2.0 ** -126]
    assert got.tolist() == want


# ---------------------------------------------------------------- budget
def test_budget_rows_golden():
    rows = []
    with open(os.path.join(HERE, "golden", "budget_rows.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(tuple(int(x) for x in line.split()))
    assert len(rows) >= 8
    for L, permille, k in rows:
        assert O.budget_rows(L, permille) == k, (L, permille)


def test_budget_is_ceil_and_clamped():
    for L in [0, 1, 7, 19, 20, 21, 999, 1000, 1001, 131072]:
        for pm in [0, 1, 25, 50, 100, 999, 1000]:
            assert O.budget_rows(L, pm) == min(L, math.ceil(L * pm / 1000 - 1e-12))


# ---------------------------------------------------------------- scores (Eq. 1)
def test_scores_one_hot_query_reads_one_column():
    rng = np.random.default_rng(1)
    d, L = 128, 50
    K = bf16_bits(rng.standard_normal((L, d)))
    for c in [0, 1, 63, 127]:
        q = np.zeros((1, d), np.float32)
        q[0, c] = 1.0
        s = O.raw_scores(bf16_bits(q), K, d ** -0.5)
        assert np.array_equal(s[0], O.bf16_bits_to_f64(K)[:, c] * d ** -0.5)


def test_scores_key_equal_to_query_gives_squared_norm():
    rng = np.random.default_rng(2)
    d = 128
    q = bf16_bits(rng.standard_normal((3, d)))
    qf = O.bf16_bits_to_f64(q)
    for g in range(3):
        s = O.raw_scores(q, q[g:g + 1], d ** -0.5)      # one key = query head g
        assert s.shape == (3, 1)
        assert math.isclose(s[g, 0], math.fsum(qf[g] ** 2) * d ** -0.5, rel_tol=1e-14)


def test_scores_brute_force_loops():
    rng = np.random.default_rng(3)
    G, L, d = 3, 9, 16
    q, K = bf16_bits(rng.standard_normal((G, d))), bf16_bits(rng.standard_normal((L, d)))
    qf, Kf = O.bf16_bits_to_f64(q).tolist(), O.bf16_bits_to_f64(K).tolist()
    s = O.raw_scores(q, K, 0.25)
    for g in range(G):
        for t in range(L):
            ref = 0.25 * math.fsum(qf[g][c] * Kf[t][c] for c in range(d))
            assert math.isclose(s[g, t], ref, rel_tol=1e-13, abs_tol=1e-15)
    # the scale multiplies, it does not divide: doubling sm_scale doubles every score
    assert np.allclose(O.raw_scores(q, K, 0.5), 2 * s, rtol=1e-15)


# ---------------------------------------------------------------- aggregation
def test_aggregate_mode0_is_max_over_group_brute():
    rng = np.random.default_rng(4)
    s = rng.standard_normal((5, 11))
    a = O.aggregate(s, O.AGG_MAX_LOGIT)
    for t in range(11):
        assert a[t] == max(s[g, t] for g in range(5))


def test_aggregate_mode1_matches_library_softmax_and_sums_to_G():
    from scipy.special import softmax
    rng = np.random.default_rng(5)
    G, L = 4, 257
    s = 3.0 * rng.standard_normal((G, L))
    a = O.aggregate(s, O.AGG_SOFTMAX_SUM)
    assert np.allclose(a, softmax(s, axis=1).sum(axis=0), rtol=1e-12)
    assert math.isclose(a.sum(), G, rel_tol=1e-12)                         # each head's softmax sums to 1
    # per-head normalisation over t (not over g): scaling one head's logits by a constant shift changes nothing
    s2 = s.copy()
    s2[2] += 7.0
    assert np.allclose(O.aggregate(s2, O.AGG_SOFTMAX_SUM), a, rtol=1e-12)


def test_modes_agree_on_ranking_when_G_is_1():
    rng = np.random.default_rng(6)
    s = rng.standard_normal((1, 500))
    for k in [1, 17, 250, 500]:
        p0 = O.topk_positions(O.aggregate(s, 0), k)
        p1 = O.topk_positions(O.aggregate(s, 1), k)
        assert np.array_equal(p0, p1)


# ---------------------------------------------------------------- top-k
def test_topk_tie_rule_and_order_by_hand():
    a = np.array([1.0, 3.0, 3.0, 2.0, 3.0])
    assert O.topk_positions(a, 0).tolist() == []
    assert O.topk_positions(a, 1).tolist() == [1]          # ties -> lower position
    assert O.topk_positions(a, 2).tolist() == [1, 2]
    assert O.topk_positions(a, 3).tolist() == [1, 2, 4]
    assert O.topk_positions(a, 4).tolist() == [1, 2, 3, 4]  # emitted ascending by position, not by score
    assert O.topk_positions(a, 5).tolist() == [0, 1, 2, 3, 4]
    assert O.topk_positions(a, 99).tolist() == [0, 1, 2, 3, 4]
    assert O.topk_positions(np.array([-1.0, -3.0, -2.0]), 2).tolist() == [0, 2]   # largest, not largest magnitude


def test_topk_brute_force_and_invariants():
    rng = np.random.default_rng(7)
    for L, k in [(1, 1), (10, 3), (1000, 50), (1000, 1000), (777, 0)]:
        a = np.round(rng.standard_normal(L), 1)       # rounding makes exact ties common
        got = O.topk_positions(a, k)
        brute = sorted(sorted(range(L), key=lambda t: (-a[t], t))[:k])
        assert got.tolist() == brute
        assert got.dtype == np.int32 and len(got) == min(k, L)
        assert np.all(np.diff(got) > 0)
        if 0 < k < L:
            rest = np.setdiff1d(np.arange(L), got)
            assert a[got].min() >= a[rest].max()


def test_select_planted_keys_tiny_hand_case():
    # L=64, d=8: every key is 0 except the planted rows, which equal q => score(planted) = |q|^2/sqrt(d) > 0 = others
    d, L, P = 8, 64, 16
    q = np.array([[1, -2, 0.5, 3, 0, 1, -1, 2]], np.float32)
    planted = [3, 17, 18, 40, 63]
    K = np.zeros((L, 1, d), np.float32)
    K[planted, 0, :] = q[0]
    k_pages = bf16_bits(K).reshape(L // P, P, 1, d)
    page_table = np.arange(L // P, dtype=np.int32)[None, :]
    sel, scores = O.select(bf16_bits(q)[None], k_pages, page_table, np.array([L]), np.array([5]), 1, d ** -0.5)
    assert sel[0][0].tolist() == planted
    assert np.allclose(scores[0][0][planted], (q ** 2).sum() / math.sqrt(d))
    # budget 100 % => identity
    sel, _ = O.select(bf16_bits(q)[None], k_pages, page_table, np.array([L]), np.array([L]), 1, d ** -0.5)
    assert sel[0][0].tolist() == list(range(L))


def test_select_uses_group_of_the_kv_head():
    # H_q=4, H_kv=2 (G=2): KV head 1 must be scored by query heads 2,3 only.
    rng = np.random.default_rng(8)
    d, L = 128, 48
    q = rng.standard_normal((1, 4, d)).astype(np.float32)
    K = rng.standard_normal((L, 2, d)).astype(np.float32)
    k_pages = bf16_bits(K).reshape(3, 16, 2, d)
    pt = np.arange(3, dtype=np.int32)[None]
    _, sc = O.select(bf16_bits(q), k_pages, pt, np.array([L]), np.array([4]), 2, 1.0)
    qf, Kf = bf16_round(q), bf16_round(K)
    for h in range(2):
        ref = np.maximum(Kf[:, h, :] @ qf[0, 2 * h], Kf[:, h, :] @ qf[0, 2 * h + 1])
        assert np.allclose(sc[0][h], ref, rtol=1e-13, atol=1e-13)


def test_select_is_invariant_to_physical_page_placement_and_ignores_tails():
    w = synth.tiny(seq_lens=(300, 77), permille=100)
    a = synth.make_inputs(w, seed=11, hostile_tails=False)
    b = synth.make_inputs(w, seed=11, spare_pages=5, hostile_tails=True)   # other page permutation + poisoned tails
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    sa, _ = O.select(synth.to_u16(a["q_rep"]), synth.to_u16(a["k_pages"]), a["page_table"].numpy(),
                     a["seq_lens"].numpy(), ks, w.n_kv_heads, 128 ** -0.5)
    # same logical content? (generators differ once spare pages change the permutation draw) -> rebuild logical view
    for inp in (a, b):
        kp, pt = synth.to_u16(inp["k_pages"]), inp["page_table"].numpy()
        sel, _ = O.select(synth.to_u16(inp["q_rep"]), kp, pt, inp["seq_lens"].numpy(), ks, w.n_kv_heads, 128 ** -0.5)
        for bb, L in enumerate(w.seq_lens):
            for h in range(w.n_kv_heads):
                rows = O.cached_rows(kp, pt, bb, L, h)
                dense = O.bf16_bits_to_f64(rows)
                q = O.bf16_bits_to_f64(synth.to_u16(inp["q_rep"]))[bb, h * w.group:(h + 1) * w.group]
                ref = (dense @ q.T).max(axis=1) * 128 ** -0.5
                want = sorted(sorted(range(L), key=lambda t: (-ref[t], t))[:ks[bb]])
                assert sel[bb][h].tolist() == want
                assert sel[bb][h].max() < L
    assert len(sa) == 2


# ---------------------------------------------------------------- gather
def test_gather_is_bitwise_index_select():
    w = synth.tiny(seq_lens=(130, 16, 5), batch=3, permille=250)
    inp = synth.make_inputs(w, seed=12, spare_pages=2)
    kp, vp, pt = synth.to_u16(inp["k_pages"]), synth.to_u16(inp["v_pages"]), inp["page_table"].numpy()
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    sel, _ = O.select(synth.to_u16(inp["q_rep"]), kp, pt, inp["seq_lens"].numpy(), ks, w.n_kv_heads, 128 ** -0.5)
    cap = max(ks) + 3
    pk, pv, pl = O.gather(kp, vp, pt, sel, cap, fill=0xBEEF)
    for b, L in enumerate(w.seq_lens):
        # dense logical view via torch ops, then library index_select
        phys = torch.as_tensor(pt[b, :(L + 15) // 16].astype(np.int64))
        dense_k = inp["k_pages"][phys].reshape(-1, w.n_kv_heads, 128)[:L]
        dense_v = inp["v_pages"][phys].reshape(-1, w.n_kv_heads, 128)[:L]
        for h in range(w.n_kv_heads):
            idx = torch.as_tensor(sel[b][h].astype(np.int64))
            assert pl[b, h] == len(idx) == ks[b]
            assert np.array_equal(pk[b, h, :len(idx)], synth.to_u16(dense_k[:, h].index_select(0, idx)))
            assert np.array_equal(pv[b, h, :len(idx)], synth.to_u16(dense_v[:, h].index_select(0, idx)))
            assert np.all(pk[b, h, len(idx):] == 0xBEEF) and np.all(pv[b, h, len(idx):] == 0xBEEF)
    assert not np.array_equal(pk, pv)


# ---------------------------------------------------------------- attention
def _attn_inputs(seed, batch=2, B=4, Hq=4, Hkv=2, n=(7, 3), cap=9, d=128, scale_q=1.0):
    rng = np.random.default_rng(seed)
    q = bf16_bits(scale_q * rng.standard_normal((batch, B, Hq, d)))
    kb, vb = bf16_bits(rng.standard_normal((batch, B, Hkv, d))), bf16_bits(rng.standard_normal((batch, B, Hkv, d)))
    pk, pv = bf16_bits(rng.standard_normal((batch, Hkv, cap, d))), bf16_bits(rng.standard_normal((batch, Hkv, cap, d)))
    pl = np.array([[n[0], n[1]]] * batch, dtype=np.int32)[:, :Hkv]
    return q, kb, vb, pk, pv, pl


def _sdpa_reference(q, kb, vb, pk, pv, pl, scale):
    """Library reference: torch SDPA in fp64 over [pool rows ; block rows], KV heads repeated G times."""
    batch, B, Hq, d = q.shape
    Hkv = kb.shape[2]
    G = Hq // Hkv
    out = np.zeros((batch, B, Hq, d))
    for b in range(batch):
        for h in range(Hkv):
            n = int(pl[b, h])
            K = torch.as_tensor(np.concatenate([O.bf16_bits_to_f64(pk[b, h, :n]), O.bf16_bits_to_f64(kb[b, :, h])]))
            V = torch.as_tensor(np.concatenate([O.bf16_bits_to_f64(pv[b, h, :n]), O.bf16_bits_to_f64(vb[b, :, h])]))
            Q = torch.as_tensor(O.bf16_bits_to_f64(q[b, :, h * G:(h + 1) * G])).permute(1, 0, 2)   # [G, B, d]
            o = torch.nn.functional.scaled_dot_product_attention(
                Q[None], K[None, None].expand(1, G, -1, -1), V[None, None].expand(1, G, -1, -1), scale=scale)
            out[b, :, h * G:(h + 1) * G] = o[0].permute(1, 0, 2).numpy()
    return out


def test_attention_matches_library_sdpa_fp64():
    args = _attn_inputs(20)
    out, lse = O.sparse_attn(*args, 128 ** -0.5)
    ref = _sdpa_reference(*args, 128 ** -0.5)
    assert out.dtype == np.float32 and out.shape == ref.shape
    assert np.allclose(out, ref, rtol=0, atol=2e-7)
    assert np.array_equal(out, ref.astype(np.float32)) or np.abs(out - ref).max() < 2e-7


def test_attention_brute_force_loops_and_lse():
    q, kb, vb, pk, pv, pl = _attn_inputs(21, batch=1, B=2, Hq=2, Hkv=1, n=(3, 0), cap=4, d=8)
    out, lse = O.sparse_attn(q, kb, vb, pk, pv, pl, 0.3)
    qf, kbf, vbf, pkf, pvf = [O.bf16_bits_to_f64(x) for x in (q, kb, vb, pk, pv)]
    for i in range(2):
        for hq in range(2):
            keys = [pkf[0, 0, j] for j in range(3)] + [kbf[0, j, 0] for j in range(2)]
            vals = [pvf[0, 0, j] for j in range(3)] + [vbf[0, j, 0] for j in range(2)]
            logit = [0.3 * math.fsum(qf[0, i, hq, c] * kk[c] for c in range(8)) for kk in keys]
            z = math.fsum(math.exp(x) for x in logit)
            for c in range(8):
                ref = math.fsum(math.exp(x) / z * v[c] for x, v in zip(logit, vals))
                assert math.isclose(out[0, i, hq, c], ref, rel_tol=2e-7, abs_tol=1e-7)
            assert math.isclose(lse[0, i, hq], math.log(z), rel_tol=1e-12)


def test_attention_closed_forms():
    d = 128
    q, kb, vb, pk, pv, pl = _attn_inputs(22, batch=1, B=2, Hq=1, Hkv=1, n=(5, 0), cap=6)
    # V == c  =>  out == c (rows of P sum to 1)
    c = bf16_bits(np.full(vb.shape, 0.75)), bf16_bits(np.full(pv.shape, 0.75))
    out, _ = O.sparse_attn(q, kb, c[0], pk, c[1], pl, d ** -0.5)
    assert np.allclose(out, 0.75, atol=1e-7)
    # all keys equal => uniform weights => out = mean of the 5 pool V rows and the 2 block V rows
    same_kb, same_pk = np.broadcast_to(kb[:, :1], kb.shape).copy(), np.broadcast_to(kb[0, 0, 0], pk.shape).copy()
    out, _ = O.sparse_attn(q, same_kb, vb, same_pk, pv, pl, d ** -0.5)
    mean = (O.bf16_bits_to_f64(pv[0, 0, :5]).sum(0) + O.bf16_bits_to_f64(vb[0, :, 0]).sum(0)) / 7
    assert np.allclose(out[0, 0, 0], mean, atol=1e-7) and np.allclose(out[0, 1, 0], mean, atol=1e-7)
    # rows beyond pool_len are ignored: poison row 5
    pk2, pv2 = pk.copy(), pv.copy()
    pk2[:, :, 5:], pv2[:, :, 5:] = bf16_bits(100.0), bf16_bits(-100.0)
    o1, _ = O.sparse_attn(q, kb, vb, pk, pv, pl, d ** -0.5)
    o2, _ = O.sparse_attn(q, kb, vb, pk2, pv2, pl, d ** -0.5)
    assert np.array_equal(o1, o2)


def test_attention_two_keys_is_a_sigmoid():
    # B=1 block key + 1 pool key: p_pool = sigmoid(l_pool - l_blk)
    d = 128
    rng = np.random.default_rng(23)
    q = bf16_bits(rng.standard_normal((1, 1, 1, d)))
    kb, vb = bf16_bits(rng.standard_normal((1, 1, 1, d))), bf16_bits(rng.standard_normal((1, 1, 1, d)))
    pk, pv = bf16_bits(rng.standard_normal((1, 1, 1, d))), bf16_bits(rng.standard_normal((1, 1, 1, d)))
    out, _ = O.sparse_attn(q, kb, vb, pk, pv, np.array([[1]]), d ** -0.5)
    qf = O.bf16_bits_to_f64(q)[0, 0, 0]
    x = d ** -0.5 * (qf @ O.bf16_bits_to_f64(pk)[0, 0, 0] - qf @ O.bf16_bits_to_f64(kb)[0, 0, 0])
    p = 1.0 / (1.0 + math.exp(-x))
    ref = p * O.bf16_bits_to_f64(pv)[0, 0, 0] + (1 - p) * O.bf16_bits_to_f64(vb)[0, 0, 0]
    assert np.allclose(out[0, 0, 0], ref, atol=1e-7)
    # single key (empty pool, B=1) => out = its V row exactly
    out, _ = O.sparse_attn(q, kb, vb, pk, pv, np.array([[0]]), d ** -0.5)
    assert np.array_equal(out[0, 0, 0], O.bf16_bits_to_f64(vb)[0, 0, 0].astype(np.float32))


def test_attention_invariant_to_pool_row_order_and_kv_head_isolation():
    q, kb, vb, pk, pv, pl = _attn_inputs(24)
    o1, _ = O.sparse_attn(q, kb, vb, pk, pv, pl, 128 ** -0.5)
    perm = np.array([3, 0, 6, 1, 5, 2, 4])
    pk2, pv2 = pk.copy(), pv.copy()
    pk2[:, 0, :7], pv2[:, 0, :7] = pk[:, 0, perm], pv[:, 0, perm]
    o2, _ = O.sparse_attn(q, kb, vb, pk2, pv2, pl, 128 ** -0.5)
    assert np.allclose(o1, o2, atol=1e-7)
    # changing KV head 1 changes only query heads 2,3 (h = hq // G, contiguous groups)
    pv3 = pv.copy()
    pv3[:, 1] = bf16_bits(np.ones(pv[:, 1].shape))
    o3, _ = O.sparse_attn(q, kb, vb, pk, pv3, pl, 128 ** -0.5)
    assert np.array_equal(o1[:, :, :2], o3[:, :, :2]) and not np.allclose(o1[:, :, 2:], o3[:, :, 2:])


def test_attention_lse_merge_identity_for_split_kv():
    # attention over [pool ; block] == LSE-weighted merge of attention over two disjoint key subsets
    q, kb, vb, pk, pv, pl = _attn_inputs(25, batch=1, B=4, Hq=2, Hkv=1, n=(8, 0), cap=8)
    full, lse = O.sparse_attn(q, kb, vb, pk, pv, pl, 128 ** -0.5)
    # part A: pool rows 0..4 + block ; part B: pool rows 5..7 + *no* block -> emulate with B keys moved into pool
    pa = np.array([[5]], dtype=np.int32)
    oa, la = O.sparse_attn(q, kb, vb, pk, pv, pa, 128 ** -0.5)
    # part B as a pure pool of rows 5..7 with a "block" that we then subtract is awkward; instead use 3 rows as block
    kb2 = pk[:, 0, 5:8][:, :, None, :]
    vb2 = pv[:, 0, 5:8][:, :, None, :]
    # query rows must match: run all 4 query rows against the 3 keys one row-block at a time
    ob = np.zeros_like(full, dtype=np.float64)
    lb = np.zeros_like(lse)
    for i in range(4):
        qi = np.broadcast_to(q[:, i:i + 1], (1, 3, 2, 128)).copy()
        o, l = O.sparse_attn(qi, kb2, vb2, pk, pv, np.array([[0]], dtype=np.int32), 128 ** -0.5)
        ob[:, i], lb[:, i] = o[:, 0], l[:, 0]
    wa, wb = np.exp(la - np.logaddexp(la, lb)), np.exp(lb - np.logaddexp(la, lb))
    merged = wa[..., None] * oa + wb[..., None] * ob
    assert np.allclose(merged, full, atol=3e-7)
    assert np.allclose(np.logaddexp(la, lb), lse, rtol=1e-12)


def test_full_budget_sparse_equals_dense_attention():
    """north_star invariant: at a 100 % budget the select->gather->sparse_attn chain equals dense
    attention over the whole prefix + block (library SDPA fp64 on the un-paged cache)."""
    w = synth.tiny(seq_lens=(90, 33), permille=1000, denoise_steps=2)
    inp = synth.make_inputs(w, seed=30, spare_pages=1, hostile_tails=True)
    kp, vp, pt = synth.to_u16(inp["k_pages"]), synth.to_u16(inp["v_pages"]), inp["page_table"].numpy()
    ks = [O.budget_rows(L, 1000) for L in w.seq_lens]
    assert ks == list(w.seq_lens)
    sel, _ = O.select(synth.to_u16(inp["q_rep"]), kp, pt, inp["seq_lens"].numpy(), ks, w.n_kv_heads, 128 ** -0.5)
    pk, pv, pl = O.gather(kp, vp, pt, sel, max(ks))
    q, kb, vb = (synth.to_u16(inp[n][0]) for n in ("q_blk", "k_blk", "v_blk"))
    out, _ = O.sparse_attn(q, kb, vb, pk, pv, pl, 128 ** -0.5)
    # dense: un-page with torch, then SDPA over [prefix ; block]
    dense_k = np.zeros((w.batch, w.n_kv_heads, max(ks), 128), np.uint16)
    dense_v = np.zeros_like(dense_k)
    for b, L in enumerate(w.seq_lens):
        phys = torch.as_tensor(pt[b, :(L + 15) // 16].astype(np.int64))
        dense_k[b, :, :L] = synth.to_u16(inp["k_pages"][phys].reshape(-1, w.n_kv_heads, 128)[:L].permute(1, 0, 2))
        dense_v[b, :, :L] = synth.to_u16(inp["v_pages"][phys].reshape(-1, w.n_kv_heads, 128)[:L].permute(1, 0, 2))
    ref = _sdpa_reference(q, kb, vb, dense_k, dense_v, np.array([[L] * w.n_kv_heads for L in w.seq_lens]), 128 ** -0.5)
    assert np.allclose(out, ref, atol=2e-7)


# ---------------------------------------------------------------- pipeline
def test_pipeline_step_is_the_sequential_composition():
    w = synth.tiny(seq_lens=(200, 64), permille=100, denoise_steps=4)
    inp = synth.make_inputs(w, seed=31)
    kp, vp, pt = synth.to_u16(inp["k_pages"]), synth.to_u16(inp["v_pages"]), inp["page_table"].numpy()
    ks = [O.budget_rows(L, w.permille) for L in w.seq_lens]
    cap = max(ks) + w.block_size
    rng = np.random.default_rng(32)
    act_k, act_v = bf16_bits(rng.standard_normal((2, 2, cap, 128))), bf16_bits(rng.standard_normal((2, 2, cap, 128)))
    act_len = np.array([[5, 9], [0, cap]], dtype=np.int32)
    layer = dict(k_pages=kp, v_pages=vp, page_table=pt, seq_lens=inp["seq_lens"].numpy(), k_per_seq=ks,
                 q_rep_next=synth.to_u16(inp["q_rep"]), q_blk=synth.to_u16(inp["q_blk"]),
                 k_blk=synth.to_u16(inp["k_blk"]), v_blk=synth.to_u16(inp["v_blk"]),
                 pool_k=act_k, pool_v=act_v, pool_len=act_len, pool_capacity=cap)
    res = O.pipeline_step([layer], w.n_attn_steps, 128 ** -0.5)[0]
    assert len(res["outs"]) == 3
    for s in range(3):
        o, _ = O.sparse_attn(layer["q_blk"][s], layer["k_blk"][s], layer["v_blk"][s], act_k, act_v, act_len, 128 ** -0.5)
        assert np.array_equal(res["outs"][s], o)
    sel, _ = O.select(layer["q_rep_next"], kp, pt, layer["seq_lens"], ks, 2, 128 ** -0.5)
    pk, pv, pl = O.gather(kp, vp, pt, sel, cap)
    assert np.array_equal(res["next_pool_k"], pk) and np.array_equal(res["next_pool_v"], pv)
    assert np.array_equal(res["next_pool_len"], pl) and pl.tolist() == [[20, 20], [7, 7]]
    # planted keys (x4 toward q_rep) are recalled by the selection
    for b in range(2):
        for h in range(2):
            planted = set(inp["planted"][b][h].tolist())
            assert len(planted & set(sel[b][h].tolist())) >= len(planted) - 1


# ---- NEXT-2: attention output of the representative query ---------------------------------------
def _rep_inputs(seed, seq_lens=(37, 5, 0), Hq=4, Hkv=2):
    w = synth.Workload("rep", len(seq_lens), tuple(seq_lens), Hq, Hkv, 16, 2, 100, "plain")
    inp = synth.make_inputs(w, seed, "cpu", spare_pages=1, hostile_tails=True, with_block_inputs=False)
    return w, (synth.to_u16(inp["q_rep"]), synth.to_u16(inp["k_pages"]), synth.to_u16(inp["v_pages"]),
               inp["page_table"].numpy(), inp["seq_lens"].numpy())


def test_rep_attn_matches_library_sdpa_and_ignores_tails():
    w, (q, kp, vp, pt, sl) = _rep_inputs(31)
    out, lse = O.rep_attn(q, kp, vp, pt, sl, w.n_kv_heads, 128 ** -0.5)
    G = w.group
    for b, L in enumerate(w.seq_lens):
        for h in range(w.n_kv_heads):
            if L == 0:
                assert np.all(out[b] == 0) and np.all(np.isneginf(lse[b]))
                continue
            K = torch.as_tensor(O.bf16_bits_to_f64(O.cached_rows(kp, pt, b, L, h)))
            V = torch.as_tensor(O.bf16_bits_to_f64(O.cached_rows(vp, pt, b, L, h)))
            Q = torch.as_tensor(O.bf16_bits_to_f64(q[b, h * G:(h + 1) * G]))                  # [G, d]
            ref = torch.nn.functional.scaled_dot_product_attention(Q[None, :, None, :], K[None, None].expand(1, G, -1, -1),
                                                                   V[None, None].expand(1, G, -1, -1), scale=128 ** -0.5)
            assert np.allclose(out[b, h * G:(h + 1) * G], ref[0, :, 0].numpy(), rtol=0, atol=1e-12)
            logits = (Q @ K.T).numpy() * 128 ** -0.5
            assert np.allclose(lse[b, h * G:(h + 1) * G], np.log(np.exp(logits).sum(axis=1)), rtol=0, atol=1e-12)


def test_rep_attn_closed_forms():
    # one cached token => its V row; constant V => that constant; the softmax weights are those of aggregate mode 1
    w, (q, kp, vp, pt, sl) = _rep_inputs(32, seq_lens=(1, 64), Hq=2, Hkv=1)
    out, _ = O.rep_attn(q, kp, vp, pt, sl, 1, 128 ** -0.5)
    v0 = O.bf16_bits_to_f64(O.cached_rows(vp, pt, 0, 1, 0))[0]
    assert np.allclose(out[0, 0], v0, atol=1e-15) and np.allclose(out[0, 1], v0, atol=1e-15)
    vp2 = vp.copy()
    vp2[:] = bf16_bits(np.float32(0.75))
    out2, _ = O.rep_attn(q, kp, vp2, pt, sl, 1, 128 ** -0.5)
    assert np.allclose(out2, 0.75, atol=1e-14)
    s = O.raw_scores(q[1], O.cached_rows(kp, pt, 1, 64, 0), 128 ** -0.5)                     # [G, 64]
    p = np.exp(s - s.max(axis=1, keepdims=True))
    p /= p.sum(axis=1, keepdims=True)
    assert np.allclose(p.sum(axis=0), O.aggregate(s, O.AGG_SOFTMAX_SUM), atol=1e-14)        # ŝ_h[s] of PAPER.md:209
    V = O.bf16_bits_to_f64(O.cached_rows(vp, pt, 1, 64, 0))
    assert np.allclose(out[1], p @ V, atol=1e-13)


# ---- NEXT-3: block-boundary cache operations ------------------------------------------------------
def test_cache_write_block_roundtrip_and_locality():
    w = synth.Workload("cw", 2, (40, 23), 4, 2, 16, 2, 100, "plain")
    inp = synth.make_inputs(w, 41, "cpu", spare_pages=2)
    kp, vp = synth.to_u16(inp["k_pages"]), synth.to_u16(inp["v_pages"])
    pt = inp["page_table"].numpy()
    rng = np.random.default_rng(3)
    k_new = rng.integers(0, 2 ** 16, size=(2, 8, 2, 128), dtype=np.uint16)
    v_new = rng.integers(0, 2 ** 16, size=(2, 8, 2, 128), dtype=np.uint16)
    pos = np.array([32, 7])                         # sequence 0: rows 32..39 (replace), sequence 1: rows 7..14 (crosses no page end... 7..14 stays in page 0)
    kp2, vp2 = O.cache_write_block(kp, vp, pt, pos, k_new, v_new)
    for b in range(2):
        for h in range(2):
            rows = O.cached_rows(kp2, pt, b, w.seq_lens[b], h)
            old = O.cached_rows(kp, pt, b, w.seq_lens[b], h)
            p0 = int(pos[b])
            assert np.array_equal(rows[p0:p0 + 8], k_new[b, :, h])                       # what was written is read back
            assert np.array_equal(rows[:p0], old[:p0]) and np.array_equal(rows[p0 + 8:], old[p0 + 8:])   # nothing else moved
            assert np.array_equal(O.cached_rows(vp2, pt, b, w.seq_lens[b], h)[p0:p0 + 8], v_new[b, :, h])
    touched = np.unique(np.nonzero((kp2 != kp).any(axis=(1, 2, 3)))[0])
    assert set(touched) <= {int(pt[0, 2]), int(pt[1, 0])}                                 # only the pages that hold those rows


def test_pool_append_block_then_attention_sees_the_rows():
    q, kb, vb, pk, pv, pl = _attn_inputs(42, batch=1, B=4, Hq=2, Hkv=1, n=(3, 0), cap=12)
    pk2, pv2, pl2 = O.pool_append_block(pk, pv, pl, kb, vb)
    assert pl2.tolist() == [[7]] and np.array_equal(pk2[0, 0, 3:7], kb[0, :, 0]) and np.array_equal(pk2[0, 0, :3], pk[0, 0, :3])
    # attention over (pool + appended block) with an EMPTY in-block set == attention over pool with that block in-block
    ref, _ = O.sparse_attn(q, kb, vb, pk, pv, pl, 0.2)
    K = np.concatenate([O.bf16_bits_to_f64(pk2[0, 0, :7])]); V = O.bf16_bits_to_f64(pv2[0, 0, :7])
    for hq in range(2):
        logits = 0.2 * O.bf16_bits_to_f64(q[0, :, hq]) @ K.T
        p = np.exp(logits - logits.max(axis=1, keepdims=True)); p /= p.sum(axis=1, keepdims=True)
        assert np.allclose(ref[0, :, hq], p @ V, atol=1e-6)


# ---------------------------------------------------------------- NEXT-4: x-query selection (reading 25)
def _xq_inputs(seed, x, batch=2, Hq=4, Hkv=2, seq_lens=(53, 16), d=128, P=16):
    rng = np.random.default_rng(seed)
    n_pages = sum((L + P - 1) // P for L in seq_lens)
    K = rng.standard_normal((n_pages, P, Hkv, d)).astype(np.float32)
    q = rng.standard_normal((batch, x, Hq, d)).astype(np.float32)
    pt = np.zeros((batch, max((L + P - 1) // P for L in seq_lens)), np.int32)
    perm, nxt = rng.permutation(n_pages), 0
    for b, L in enumerate(seq_lens):
        for j in range((L + P - 1) // P):
            pt[b, j] = perm[nxt]
            nxt += 1
    return bf16_bits(q), bf16_bits(K), pt, np.array(seq_lens)


def test_select_xq_with_one_query_is_select():
    q, K, pt, L = _xq_inputs(31, 1)
    sa, sca = O.select_xq(q, K, pt, L, [7, 3], 2, 128 ** -0.5)
    sb, scb = O.select(q[:, 0], K, pt, L, [7, 3], 2, 128 ** -0.5, O.AGG_MAX_LOGIT)
    for b in range(2):
        for h in range(2):
            assert sa[b][h].tolist() == sb[b][h].tolist() and np.array_equal(sca[b][h], scb[b][h])


def test_select_xq_brute_force_loops():
    # a[t] = max_j max_g scale * q[j, h*G+g] . K[t, h], written as scalar loops over widened values
    x, G, d = 3, 2, 128
    q, K, pt, L = _xq_inputs(32, x, seq_lens=(21, 5))
    qf, Kf = O.bf16_bits_to_f64(q), O.bf16_bits_to_f64(K)
    sel, sc = O.select_xq(q, K, pt, L, [4, 5], 2, 0.25)
    for b in range(2):
        for h in range(2):
            ref = []
            for t in range(int(L[b])):
                krow = Kf[pt[b, t // 16], t % 16, h]
                best = -math.inf
                for j in range(x):
                    for g in range(G):
                        acc = 0.0
                        for c in range(d):
                            acc += qf[b, j, h * G + g, c] * krow[c]
                        best = max(best, 0.25 * acc)
                ref.append(best)
            assert np.allclose(sc[b][h], ref, rtol=1e-12, atol=1e-12)
            k = min([4, 5][b], int(L[b]))
            want = sorted(sorted(range(int(L[b])), key=lambda t: (-ref[t], t))[:k])
            assert sel[b][h].tolist() == want


def test_select_xq_invariants():
    x = 4
    q, K, pt, L = _xq_inputs(33, x)
    _, sc = O.select_xq(q, K, pt, L, [5, 5], 2, 1.0)
    # the order of the x queries does not matter
    _, sc_perm = O.select_xq(q[:, ::-1].copy(), K, pt, L, [5, 5], 2, 1.0)
    # a duplicated query changes nothing; one more query never lowers a score; a subset never raises one
    _, sc_dup = O.select_xq(np.concatenate([q, q[:, :1]], axis=1), K, pt, L, [5, 5], 2, 1.0)
    _, sc_sub = O.select_xq(q[:, :2].copy(), K, pt, L, [5, 5], 2, 1.0)
    singles = [O.select(q[:, j].copy(), K, pt, L, [5, 5], 2, 1.0)[1] for j in range(x)]
    for b in range(2):
        for h in range(2):
            assert np.array_equal(sc[b][h], sc_perm[b][h]) and np.array_equal(sc[b][h], sc_dup[b][h])
            assert np.all(sc_sub[b][h] <= sc[b][h])
            # and it is exactly the pointwise maximum of the x single-query score planes
            assert np.array_equal(sc[b][h], np.max([singles[j][b][h] for j in range(x)], axis=0))


def test_select_xq_planted_key_found_by_the_one_query_that_matches():
    # keys are 0 except one row equal to query j=2's head 1; every other query is orthogonal noise on other channels
    d, L, P, x = 128, 32, 16, 4
    q = np.zeros((1, x, 2, d), np.float32)
    for j in range(x):
        q[0, j, :, 8 * j:8 * j + 8] = -1.0          # negative everywhere it is non-zero: only the planted row scores > 0 ...
    q[0, 2, 1, 100:108] = 2.0
    K = np.zeros((L, 1, d), np.float32)
    K[19, 0, 100:108] = 2.0                          # ... and only through query 2, head 1
    k_pages = bf16_bits(K).reshape(L // P, P, 1, d)
    pt = np.arange(L // P, dtype=np.int32)[None]
    sel, sc = O.select_xq(bf16_bits(q), k_pages, pt, np.array([L]), [1], 1, 1.0)
    assert sel[0][0].tolist() == [19] and sc[0][0][19] == 32.0 and np.all(np.delete(sc[0][0], 19) == 0.0)
