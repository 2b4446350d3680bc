"""Helpers shared by the GPU parity tests: run the CUDA path through the C-ABI binding and the
oracle on the same seeded inputs, and compare under the tolerances of BASELINE.json's north_star."""
import numpy as np
import torch

from oracle import herald_oracle as O
from paper_2606_21633_b200 import synth

REL_BAND = 1e-3     # north_star: index sets exact except keys within 1e-3 relative of the k-th score
ABS_FLOOR = 1e-6    # DESIGN.md reading 8: absolute floor for a_k ~ 0
ATTN_TOL = 2e-3     # north_star: attention output max abs error <= 2e-3


def check_selection(sel_gpu, cnt_gpu, scores_oracle, k, L, tag=""):
    """sel_gpu: int array (first cnt_gpu entries valid). Returns number of positions differing from the oracle set."""
    kk = min(k, L)
    assert cnt_gpu == kk, f"{tag}: sel_cnt {cnt_gpu} != {kk}"
    s = np.asarray(sel_gpu[:kk], dtype=np.int64)
    if kk == 0:
        return 0
    assert s.min() >= 0 and s.max() < L, f"{tag}: index out of range"
    assert np.all(np.diff(s) > 0), f"{tag}: indices not strictly ascending / not unique"
    want = O.topk_positions(scores_oracle, kk).astype(np.int64)
    if np.array_equal(s, want):
        return 0
    a = scores_oracle
    a_k = np.sort(a)[::-1][kk - 1]
    band = REL_BAND * abs(a_k) + ABS_FLOOR
    must = np.nonzero(a > a_k + band)[0]
    missing = np.setdiff1d(must, s)
    assert missing.size == 0, f"{tag}: {missing.size} keys above the band are missing, e.g. {missing[:5]}"
    low = s[a[s] < a_k - band]
    assert low.size == 0, f"{tag}: {low.size} selected keys lie below the band, e.g. {low[:5]}"
    return int(np.setdiff1d(s, want).size)


def oracle_inputs(inp):
    return dict(k_pages=synth.to_u16(inp["k_pages"]), v_pages=synth.to_u16(inp["v_pages"]),
                page_table=inp["page_table"].cpu().numpy(), seq_lens=inp["seq_lens"].cpu().numpy(),
                q_rep=synth.to_u16(inp["q_rep"]))
