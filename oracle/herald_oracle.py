"""HERALD per-block sparse-KV hot path -- the CPU ORACLE (test infrastructure only).

This file is TEST INFRASTRUCTURE.  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it.
The product path (``paper_2606_21633_b200``) never imports, links or calls
anything in ``oracle/``, and this file imports nothing from the product.

It is a plain, slow, fp64 NumPy restatement of what the hot path computes,
written from /root/reference/PAPER.md (HERALD, arxiv/paper_2606_21633) and the
readings listed in DESIGN.md ("Readings of the paper").  There is no blocking,
fusion or reordering beyond what each definition states; a library primitive
(``@`` matmul, ``np.lexsort``, ``np.exp``) serves as a step.

Citations are ``PAPER.md:<line>`` plus the section / equation they fall in.

Data conventions (same as include/herald.h, but HOST NumPy arrays):
  * bf16 tensors are ``uint16`` arrays holding the bf16 bit patterns; they are
    widened exactly to fp64 (bf16 -> fp32 is a 16-bit shift; fp32 -> fp64 is exact).
  * the K/V cache is paged: ``k_pages[n_pages, page_size, H_kv, d]``, with
    ``page_table[batch, max_pages]`` (logical page -> physical page) and
    ``seq_lens[batch]``; token t of sequence b lives at page ``page_table[b, t // page_size]``,
    slot ``t % page_size`` (section V: "paged KV cache management").
  * query head ``hq`` belongs to KV head ``hq // G`` with ``G = H_q // H_kv``
    (section IV-B4: "G is the number of query heads that share one KV head under GQA").

Pin status (see tests/test_oracle_pins.py, all ``-m "not gpu"``; ``rep_attn``, ``cache_write_block`` and ``pool_append_block`` included): every function
below is pinned against something other than itself -- closed forms, brute
force pure-Python loops, library SDPA / softmax, invariants.  ``select_xq`` is
"parity unpinned" AGAINST THE PAPER: PAPER.md:137 (Fig. 8) and :161 sweep the
query count x of the selection kernel but never say how the x queries' scores
combine into one ranking, so the function follows DESIGN.md reading 25 (the
maximum over the x queries, as mode 0 takes it over the G heads); its
arithmetic under that reading is pinned like the rest (x = 1 reduces to
``select``, brute force loops, permutation and monotonicity invariants).
"""
from __future__ import annotations

import numpy as np

AGG_MAX_LOGIT = 0     # BASELINE.json north_star: max over the group's query heads of q.k/sqrt(d)
AGG_SOFTMAX_SUM = 1   # PAPER.md:209 section IV-B4: s^_h[s] = sum_g exp(s[g,s] - m_g) / l_g


# ----------------------------------------------------------------------------
# bf16 <-> fp64
# ----------------------------------------------------------------------------
def bf16_bits_to_f64(u16: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns (uint16) to fp64."""
    u16 = np.ascontiguousarray(u16, dtype=np.uint16)
    f32 = (u16.astype(np.uint32) << np.uint32(16)).view(np.float32)
    return f32.astype(np.float64)


# ----------------------------------------------------------------------------
# budget (reading 5)
# ----------------------------------------------------------------------------
def budget_rows(seq_len: int, permille: int) -> int:
    """k_b = min(L_b, ceil(rho * L_b)) with rho = permille / 1000, in integers.

    PAPER.md:201 (section IV-B4): "k is the per-KV-head selection budget";
    PAPER.md:227 (Table I): budgets are given as a % of the KV cache.
    BASELINE.json fixes the rounding: 5 % of 4096 -> 205, 5 % of 32768 -> 1639 (ceil).
    """
    seq_len = int(seq_len)
    permille = int(permille)
    assert seq_len >= 0 and 0 <= permille <= 1000
    return min(seq_len, (seq_len * permille + 999) // 1000)


# ----------------------------------------------------------------------------
# paged cache access
# ----------------------------------------------------------------------------
def cached_rows(pages_u16: np.ndarray, page_table: np.ndarray, b: int, seq_len: int, h: int) -> np.ndarray:
    """The ``seq_len`` cached rows (bf16 bits, [seq_len, d]) of sequence b, KV head h,
    in logical token order, read through the page table.  Tail slots of the last
    page (t >= seq_len) are never read (reading 18)."""
    page_size = pages_u16.shape[1]
    t = np.arange(seq_len, dtype=np.int64)
    phys = page_table[b, t // page_size].astype(np.int64)
    slot = t % page_size
    return pages_u16[phys, slot, h, :]


# ----------------------------------------------------------------------------
# step 1: scores  (Eq.(1); section IV-B4 "raw attention scores s[g,s]")
# ----------------------------------------------------------------------------
def raw_scores(q_rep_u16: np.ndarray, k_rows_u16: np.ndarray, sm_scale: float) -> np.ndarray:
    """s[g, t] = sm_scale * sum_c q[g, c] * K[t, c]   for the G query heads of one KV head.

    q_rep_u16: [G, d] bf16 bits (the representative query's heads of this group,
    post-RoPE -- DESIGN.md reading 3);  k_rows_u16: [L, d] bf16 bits.  Returns fp64 [G, L].
    Eq.(1) has no 1/sqrt(d); the kernel is FlashAttention-style
     and BASELINE.json's north_star says q.k/sqrt(d): sm_scale = d**-0.5
    is passed by the caller (reading 2)."""
    q = bf16_bits_to_f64(q_rep_u16)          # [G, d]
    k = bf16_bits_to_f64(k_rows_u16)         # [L, d]
    return float(sm_scale) * (q @ k.T)       # [G, L]


# ----------------------------------------------------------------------------
# step 2: aggregation over the GQA group
# ----------------------------------------------------------------------------
def aggregate(s: np.ndarray, agg_mode: int) -> np.ndarray:
    """One importance value per cached position from the G per-head scores s[g, t].

    mode 0 (north_star): a[t] = max_g s[g, t].
    mode 1: m_g = max_t s[g,t];  l_g = sum_t exp(s[g,t] - m_g);
                           a[t] = sum_g exp(s[g,t] - m_g) / l_g.
    """
    G, L = s.shape
    if L == 0:
        return np.zeros((0,), dtype=np.float64)
    if agg_mode == AGG_MAX_LOGIT:
        return s.max(axis=0)
    if agg_mode == AGG_SOFTMAX_SUM:
        m = s.max(axis=1, keepdims=True)                 # m_g
        e = np.exp(s - m)
        l = e.sum(axis=1, keepdims=True)                 # l_g
        return (e / l).sum(axis=0)
    raise ValueError("agg_mode must be 0 or 1")


# ----------------------------------------------------------------------------
# step 3: top-k  ("a single min-heap top-k pass extracts the k most attended positions")
# ----------------------------------------------------------------------------
def topk_positions(a: np.ndarray, k: int) -> np.ndarray:
    """The k positions of largest a[t]; ties -> lower position; emitted ascending
    (reading 7).  Full sort of (a descending, t ascending), keep the first k."""
    L = a.shape[0]
    k = min(int(k), L)
    assert np.all(np.isfinite(a)), "non-finite scores are undefined (DESIGN.md reading 19)"
    t = np.arange(L, dtype=np.int64)
    order = np.lexsort((t, -a))            # primary key: -a ascending (= a descending); secondary: t ascending
    keep = order[:k]
    return np.sort(keep).astype(np.int32)


def select(q_rep_u16, k_pages_u16, page_table, seq_lens, k_per_seq, n_kv_heads, sm_scale, agg_mode=AGG_MAX_LOGIT):
    """Representative-query selection for every (sequence b, KV head h).

    PAPER.md:141-163 (section IV-A2): one representative query replaces the B queries;
    "the CPU still scores every entry in the full prefix KV cache".
    q_rep_u16: [batch, H_q, d].  Returns (sel, scores):
      sel[b][h]    int32 ascending positions, len = min(k_per_seq[b], seq_lens[b])
      scores[b][h] fp64 [L_b] aggregated importance a[t].
    """
    batch, H_q, d = q_rep_u16.shape
    G = H_q // n_kv_heads
    assert G * n_kv_heads == H_q
    sel, scores = [], []
    for b in range(batch):
        L = int(seq_lens[b])
        sel_b, sc_b = [], []
        for h in range(n_kv_heads):
            k_rows = cached_rows(k_pages_u16, page_table, b, L, h)
            s = raw_scores(q_rep_u16[b, h * G:(h + 1) * G, :], k_rows, sm_scale)
            a = aggregate(s, agg_mode)
            sel_b.append(topk_positions(a, int(k_per_seq[b])))
            sc_b.append(a)
        sel.append(sel_b)
        scores.append(sc_b)
    return sel, scores


# ----------------------------------------------------------------------------
# step 4: gather  ("gathers the selected entries into a contiguous ... buffer")
# ----------------------------------------------------------------------------
def gather(k_pages_u16, v_pages_u16, page_table, sel, pool_capacity, fill=0):
    """pool_K[b, h, j, :] = K[b, sel[b][h][j], h, :] (bit copies), same for V; row j is
    the j-th selected position in ascending order.  Rows j >= len(sel[b][h]) keep ``fill``.
    Returns (pool_k, pool_v, pool_len) with pools uint16 [batch, H_kv, pool_capacity, d]."""
    batch = len(sel)
    H_kv = k_pages_u16.shape[2]
    d = k_pages_u16.shape[3]
    page_size = k_pages_u16.shape[1]
    pool_k = np.full((batch, H_kv, pool_capacity, d), fill, dtype=np.uint16)
    pool_v = np.full((batch, H_kv, pool_capacity, d), fill, dtype=np.uint16)
    pool_len = np.zeros((batch, H_kv), dtype=np.int32)
    for b in range(batch):
        for h in range(H_kv):
            pos = np.asarray(sel[b][h], dtype=np.int64)
            n = pos.shape[0]
            assert n <= pool_capacity
            phys = page_table[b, pos // page_size].astype(np.int64)
            slot = pos % page_size
            pool_k[b, h, :n, :] = k_pages_u16[phys, slot, h, :]
            pool_v[b, h, :n, :] = v_pages_u16[phys, slot, h, :]
            pool_len[b, h] = n
    return pool_k, pool_v, pool_len


# ----------------------------------------------------------------------------
# step 5: denoising attention over critical KV + in-block KV
# ("tokens attend bidirectionally within the current block and causally to the
#  cached KV"; "The main stream denoises block n using the KV cache in the active sparse pool")
# ----------------------------------------------------------------------------
def sparse_attn(q_blk_u16, k_blk_u16, v_blk_u16, pool_k_u16, pool_v_u16, pool_len, sm_scale):
    """O[b,i,hq,:] = softmax_j(sm_scale * Q[b,i,hq,:].K'_j) . V'_j over
    K' = pool_K[b,h,0:n_bh] followed by K_blk[b,0:B,h]  (h = hq // G); no mask: the pool
    is prefix, the block is bidirectional (readings 11, 12).

    q_blk_u16 [batch,B,H_q,d]; k_blk/v_blk [batch,B,H_kv,d]; pools [batch,H_kv,cap,d];
    pool_len [batch,H_kv].  Returns (out fp32 [batch,B,H_q,d] rounded once from fp64,
    lse fp64 [batch,B,H_q] = log sum_j exp(logit_j))."""
    batch, B, H_q, d = q_blk_u16.shape
    H_kv = k_blk_u16.shape[2]
    G = H_q // H_kv
    out = np.zeros((batch, B, H_q, d), dtype=np.float32)
    lse = np.zeros((batch, B, H_q), dtype=np.float64)
    for b in range(batch):
        for h in range(H_kv):
            n = int(pool_len[b, h])
            Kp = np.concatenate([bf16_bits_to_f64(pool_k_u16[b, h, :n, :]),
                                 bf16_bits_to_f64(k_blk_u16[b, :, h, :])], axis=0)   # [n+B, d]
            Vp = np.concatenate([bf16_bits_to_f64(pool_v_u16[b, h, :n, :]),
                                 bf16_bits_to_f64(v_blk_u16[b, :, h, :])], axis=0)
            for g in range(G):
                hq = h * G + g
                Q = bf16_bits_to_f64(q_blk_u16[b, :, hq, :])            # [B, d]
                logits = float(sm_scale) * (Q @ Kp.T)                   # [B, n+B]
                m = logits.max(axis=1, keepdims=True)
                p = np.exp(logits - m)
                z = p.sum(axis=1, keepdims=True)
                out[b, :, hq, :] = ((p @ Vp) / z).astype(np.float32)
                lse[b, :, hq] = (m + np.log(z))[:, 0]
    return out, lse


# ----------------------------------------------------------------------------
# step 6: one block step of the dual-stream pipeline
# (section IV-B1; Fig. 11)
# ----------------------------------------------------------------------------
def pipeline_step(layers, n_steps, sm_scale, agg_mode=AGG_MAX_LOGIT):
    """Sequential composition the overlapped pipeline must equal (the
    retrieval stream "affects only the selection and never the generated output"):

      main stream      : for step in 0..n_steps-1, for each layer: sparse_attn over the ACTIVE pool
      retrieval stream : for each layer: select with q_rep_next, gather into the IDLE pool
      then swap active / idle ("the two pool pointers are swapped at every block transition").

    ``layers`` is a list of dicts with keys: k_pages, v_pages, page_table, seq_lens, k_per_seq,
    q_rep_next [batch,H_q,d], q_blk/k_blk/v_blk [n_steps, ...], pool_k/pool_v/pool_len (ACTIVE), pool_capacity.
    Returns per layer: dict(outs=[n_steps] fp32 arrays, next_pool_k, next_pool_v, next_pool_len, sel).
    """
    results = []
    for ly in layers:
        outs = []
        for s in range(n_steps):
            o, _ = sparse_attn(ly["q_blk"][s], ly["k_blk"][s], ly["v_blk"][s],
                               ly["pool_k"], ly["pool_v"], ly["pool_len"], sm_scale)
            outs.append(o)
        H_kv = ly["k_pages"].shape[2]
        sel, _ = select(ly["q_rep_next"], ly["k_pages"], ly["page_table"], ly["seq_lens"],
                        ly["k_per_seq"], H_kv, sm_scale, agg_mode)
        pk, pv, pl = gather(ly["k_pages"], ly["v_pages"], ly["page_table"], sel, ly["pool_capacity"])
        results.append(dict(outs=outs, next_pool_k=pk, next_pool_v=pv, next_pool_len=pl, sel=sel))
    return results


# ----------------------------------------------------------------------------
# NEXT-2: attention output of the representative query itself
# (section IV-B4: the fused kernel "maintains the FlashAttention statistics (m_g, l_g, o_g)"
#  next to the raw scores; the output o_g goes back to the GPU for the layer's FFN)
# ----------------------------------------------------------------------------
def rep_attn(q_rep_u16, k_pages_u16, v_pages_u16, page_table, seq_lens, n_kv_heads, sm_scale):
    """o[b, hq, :] = softmax_t(sm_scale * q_rep[b, hq] . K[b, t, h]) . V[b, t, h, :] over every cached t < seq_lens[b]
    (h = hq // G), the plain definition.  Returns (out fp64 [batch, H_q, d], lse fp64 [batch, H_q]); a sequence with no
    cached token gives out = 0 and lse = -inf."""
    batch, H_q, d = q_rep_u16.shape
    G = H_q // n_kv_heads
    out = np.zeros((batch, H_q, d), dtype=np.float64)
    lse = np.full((batch, H_q), -np.inf, dtype=np.float64)
    for b in range(batch):
        L = int(seq_lens[b])
        if L == 0:
            continue
        for h in range(n_kv_heads):
            K = bf16_bits_to_f64(cached_rows(k_pages_u16, page_table, b, L, h))      # [L, d]
            V = bf16_bits_to_f64(cached_rows(v_pages_u16, page_table, b, L, h))
            s = raw_scores(q_rep_u16[b, h * G:(h + 1) * G, :], cached_rows(k_pages_u16, page_table, b, L, h), sm_scale)   # [G, L]
            m = s.max(axis=1, keepdims=True)
            p = np.exp(s - m)
            z = p.sum(axis=1, keepdims=True)
            out[b, h * G:(h + 1) * G, :] = (p @ V) / z
            lse[b, h * G:(h + 1) * G] = (m + np.log(z))[:, 0]
            del K
    return out, lse


# ----------------------------------------------------------------------------
# NEXT-3: block-boundary cache operations
# (the draft KV of block n is "appended temporarily" to the full KV pool; at the end of
#  the block the true KV is "written to both block n+1's GPU pool and the full KV pool, replacing the draft")
# ----------------------------------------------------------------------------
def cache_write_block(k_pages_u16, v_pages_u16, page_table, write_pos, k_new_u16, v_new_u16):
    """K[b, write_pos[b] + i, h, :] = k_new[b, i, h, :] for i < B (same for V), through the page table: appends the B
    rows of a block (draft or true) at logical position write_pos[b], or replaces rows already there.  Bit copies, in
    place on copies of the page arrays, which are returned."""
    kp, vp = k_pages_u16.copy(), v_pages_u16.copy()
    page_size = kp.shape[1]
    batch, B = k_new_u16.shape[0], k_new_u16.shape[1]
    for b in range(batch):
        for i in range(B):
            t = int(write_pos[b]) + i
            phys, slot = int(page_table[b, t // page_size]), t % page_size
            kp[phys, slot] = k_new_u16[b, i]
            vp[phys, slot] = v_new_u16[b, i]
    return kp, vp


def pool_append_block(pool_k_u16, pool_v_u16, pool_len, k_new_u16, v_new_u16):
    """pool[b, h, pool_len[b, h] + i, :] = k_new[b, i, h, :] for i < B, then pool_len += B (the completed block joins the
    next block's pool; reading 10 of DESIGN.md: pool_capacity >= k + B).  Returns copies."""
    pk, pv, pl = pool_k_u16.copy(), pool_v_u16.copy(), np.array(pool_len, dtype=np.int32).copy()
    batch, H_kv, cap, _ = pk.shape
    B = k_new_u16.shape[1]
    for b in range(batch):
        for h in range(H_kv):
            n = int(pl[b, h])
            assert n + B <= cap
            pk[b, h, n:n + B] = k_new_u16[b, :, h]
            pv[b, h, n:n + B] = v_new_u16[b, :, h]
            pl[b, h] = n + B
    return pk, pv, pl


# ----------------------------------------------------------------------------
# NEXT-4: selection with x queries  (PAPER.md:137 Fig. 8, :143, :161 -- parity unpinned against the paper, see header)
# ----------------------------------------------------------------------------
def select_xq(q_x_u16, k_pages_u16, page_table, seq_lens, k_per_seq, n_kv_heads, sm_scale):
    """Selection scored by x queries per sequence instead of one ("B queries perform attention in GEMM
    form"; :161: the cost "shrink[s] in proportion to the query count"; Fig. 8 sweeps x from B = 32 down to 1).

    q_x_u16: [batch, x, H_q, d] bf16 bits.  DESIGN.md reading 25 (the paper does not define the combination):
        a[t] = max over the x queries j and the G heads g of the group of  sm_scale * q_x[b, j, h*G+g] . K[b, t, h]
    i.e. mode 0 of ``aggregate`` taken over all x*G score rows; then the same top-k.  Returns (sel, scores) like ``select``.
    """
    batch, x, H_q, d = q_x_u16.shape
    G = H_q // n_kv_heads
    assert G * n_kv_heads == H_q and x >= 1
    sel, scores = [], []
    for b in range(batch):
        L = int(seq_lens[b])
        sel_b, sc_b = [], []
        for h in range(n_kv_heads):
            k_rows = cached_rows(k_pages_u16, page_table, b, L, h)
            rows = [raw_scores(q_x_u16[b, j, h * G:(h + 1) * G, :], k_rows, sm_scale) for j in range(x)]   # x arrays [G, L]
            a = aggregate(np.concatenate(rows, axis=0), AGG_MAX_LOGIT)
            sel_b.append(topk_positions(a, int(k_per_seq[b])))
            sc_b.append(a)
        sel.append(sel_b)
        scores.append(sc_b)
    return sel, scores
