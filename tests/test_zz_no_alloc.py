"""herald_select_static: herald_select with its workspace in a file-scope __device__ array of the library, for callers
that may not allocate (include/herald.h).  Collected last on purpose (the suite runs with pytest -x).

The GPU test compares the new entry point with the existing path -- same kernels, same inputs, so the index sets must be
identical, bit for bit (the bar the other selection tests use for integer work) -- on calls in a row that share the
array: a larger shape first, then a smaller one whose scratch region holds the first call's leftovers, then the first
again."""
import numpy as np
import pytest
import torch

from oracle import herald_oracle as O
from paper_2606_21633_b200 import synth
from parity_util import check_selection, oracle_inputs


@pytest.fixture(scope="module")
def H():
    from paper_2606_21633_b200 import build
    build.build()
    from paper_2606_21633_b200 import herald
    return herald


def test_static_scratch_limit_is_stated_and_enforced_before_any_cuda_call(H):
    assert H.herald_select_static_max_bytes() == 16 << 20
    fits = H.make_shape(8, 28, 4, 32, 32768, 2048, 1671)            # C2: 4.5 MiB
    assert H.herald_select_workspace_bytes(fits) <= H.herald_select_static_max_bytes()
    big = H.make_shape(16, 32, 8, 16, 65536, 4096, 3293)            # C4: 34 MiB
    assert H.herald_select_workspace_bytes(big) > H.herald_select_static_max_bytes()
    cache = H.Cache(0x1000, 0x1000, 16 * 8 * 128, 8 * 128, 128, 0x1000, 0x1000)
    with pytest.raises(H.HeraldError) as e:
        H.herald_select_static(big, cache, 0x1000, 0x1000, 0x1000, 0x1000, stream=0)
    assert e.value.code == H.ERR_WORKSPACE_TOO_SMALL and "herald_select_static" in str(e.value)


CASES = [
    ("g7_ragged", synth.Workload("g7", 3, (5000, 3333, 16), 28, 4, 32, 4, 50, "planted", 20), 2, True),
    ("tiny_ragged", synth.tiny(seq_lens=(300, 77), permille=100), 3, True),
    ("C1", synth.config("C1"), 0, False),
]


def _both_paths(H, dev, w, inp, ks):
    cap = max(max(ks), 1) + w.block_size
    max_seq = (w.max_seq_len + 15) // 16 * 16
    shape = H.make_shape(w.batch, w.n_q_heads, w.n_kv_heads, w.block_size, max_seq, inp["page_table"].shape[1], cap)
    cache = H.make_cache(inp["k_pages"], inp["v_pages"], inp["page_table"], inp["seq_lens"])
    k_per_seq = torch.tensor(ks, dtype=torch.int32, device=dev)
    out = {}
    for name in ("existing", "static"):
        sel_idx = torch.full((w.batch, w.n_kv_heads, cap), -7, dtype=torch.int32, device=dev)
        sel_cnt = torch.full((w.batch, w.n_kv_heads), -7, dtype=torch.int32, device=dev)
        if name == "existing":
            ws = H.alloc_workspace(H.herald_select_workspace_bytes(shape), dev)
            H.herald_select(shape, cache, inp["q_rep"], k_per_seq, sel_idx, sel_cnt, None, ws)
        else:
            H.herald_select_static(shape, cache, inp["q_rep"], k_per_seq, sel_idx, sel_cnt)
        torch.cuda.synchronize()
        out[name] = (sel_idx.cpu().numpy(), sel_cnt.cpu().numpy())
    return out


@pytest.mark.gpu
def test_select_static_equals_select_on_calls_in_a_row(H, cuda):
    prepared = []
    for name, w, spare, hostile in CASES:
        inp = synth.make_inputs(w, seed=500 + len(name), device=cuda, spare_pages=spare, hostile_tails=hostile)
        ks = [H.herald_budget_rows(L, w.permille) for L in w.seq_lens]
        prepared.append((name, w, inp, ks))
    first = {}
    for rnd in range(2):                        # every shape twice: each call finds another call's leftovers in the array
        for name, w, inp, ks in prepared:
            got = _both_paths(H, cuda, w, inp, ks)
            (idx_e, cnt_e), (idx_s, cnt_s) = got["existing"], got["static"]
            assert np.array_equal(cnt_s, cnt_e), (name, rnd)
            assert np.array_equal(idx_s, idx_e), (name, rnd, "index sets differ from herald_select's")
            assert cnt_s.min() >= 0 and np.all(idx_s[..., -1] == -7), "entries past sel_cnt must stay untouched"
            if rnd == 0:
                first[name] = (idx_s, cnt_s)
            else:
                assert np.array_equal(idx_s, first[name][0]) and np.array_equal(cnt_s, first[name][1]), (name, "not repeatable")
    # and against the oracle, like the existing path's own parity test (north_star's tie band)
    name, w, inp, ks = prepared[0]
    oi = oracle_inputs(inp)
    _, sc_o = O.select(oi["q_rep"], oi["k_pages"], oi["page_table"], oi["seq_lens"], ks, w.n_kv_heads, 128 ** -0.5, 0)
    idx_s, cnt_s = first[name]
    differing = 0
    for b, L in enumerate(w.seq_lens):
        for h in range(w.n_kv_heads):
            differing += check_selection(idx_s[b, h], int(cnt_s[b, h]), sc_o[b][h], ks[b], L, f"static {name} b{b} h{h}")
    assert differing <= max(1, w.batch * w.n_kv_heads // 4)
