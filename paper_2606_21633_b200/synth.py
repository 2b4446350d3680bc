"""Seeded synthetic inputs for the HERALD hot path (shared by tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic: no scores, no top-k, no budget
rounding, no softmax.  It only draws tensors with the shapes, value distributions and
structure of BASELINE.json's configs (stand-ins for the paper's LongBench-driven
workloads, which are not available here -- see DESIGN.md "Input recipe"):

  * Q, K, V: bf16 round-to-nearest of i.i.d. N(0,1) draws from a seeded torch generator;
  * "planted" heavy-hitter keys: row = bf16(eps + 4 * q_hat), q_hat = q_rep[b, h*G+g*] / |.|,
    g* = planted ordinal mod G, positions a seeded sample without replacement per (b, h);
  * "zipf" key-norm profile: K[t] = eps_t * (1 + 7 / r_t), r_t a seeded random permutation of 1..L_b;
  * paged cache [n_pages, page_size, H_kv, d] with a seeded random page permutation
    (identity for config C1), optional never-referenced spare pages and hostile tail slots.

It imports neither the CUDA binding nor anything under ``oracle/``.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional

import torch

PAGE_SIZE = 16
HEAD_DIM = 128


@dataclass(frozen=True)
class Workload:
    name: str
    batch: int
    seq_lens: tuple            # one entry per sequence
    n_q_heads: int
    n_kv_heads: int
    block_size: int            # B
    denoise_steps: int         # T ; the block step runs T-1 attention steps
    permille: int              # KV budget in 1/1000 of the context (50 = 5 %)
    structure: str = "plain"   # "plain" | "planted" | "zipf"
    planted_per_unit: int = 0
    identity_pages: bool = False
    n_layers: int = 1
    head_dim: int = HEAD_DIM
    page_size: int = PAGE_SIZE

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def max_seq_len(self) -> int:
        return max(self.seq_lens) if len(self.seq_lens) else 0

    @property
    def n_attn_steps(self) -> int:
        return self.denoise_steps - 1


def config(name: str) -> Workload:
    """BASELINE.json ``configs`` C1..C5 (one layer's inputs per make_inputs call; C5 draws one set per layer)."""
    if name == "C1":   # single layer, 1 sequence, L=4096, 4/1 heads, B=16, T=8, 5 %, 32 planted keys
        return Workload("C1", 1, (4096,), 4, 1, 16, 8, 50, "planted", 32, identity_pages=True)
    if name == "C2":   # Qwen2.5-7B-shaped layer: 28/4, batch 8 x 32768, B=32, T=16, 5 %, 0.5 % planted
        return Workload("C2", 8, (32768,) * 8, 28, 4, 32, 16, 50, "planted", 164)
    if name == "C3":   # long context: batch 4 x 131072, 28/4, B=32, T=16, 5 %
        return Workload("C3", 4, (131072,) * 4, 28, 4, 32, 16, 50, "plain")
    if name.startswith("C4"):  # Qwen3-8B-shaped: 32/8, batch 16 x 65536, B=16, T=8, budgets 2.5/5/10 %
        permille = {"C4": 50, "C4@2.5": 25, "C4@5": 50, "C4@10": 100}[name]
        return Workload(name, 16, (65536,) * 16, 32, 8, 16, 8, permille, "zipf")
    if name.startswith("C5"):  # 28-layer stack (28/4/128), batch 32, ragged contexts U{8192..131072}, B=32, T=16, 5 %
        n_layers = int(name[3:]) if name.startswith("C5x") else 28      # "C5x4" = the same stack cut to 4 layers
        gen = torch.Generator(device="cpu")
        gen.manual_seed(21633 + 5006)          # fixed draw: mean context 66.8 K tokens, 4.3 GB of K+V per layer
        lens = torch.randint(8192, 131073, (32,), generator=gen)
        return Workload(name, 32, tuple(int(x) for x in lens), 28, 4, 32, 16, 50, "plain", n_layers=n_layers)
    raise KeyError(name)


def tiny(name="tiny", batch=2, seq_lens=(300, 77), n_q_heads=4, n_kv_heads=2, block_size=16,
         denoise_steps=3, permille=100, structure="planted", planted_per_unit=5) -> Workload:
    """Small ragged case spanning several pages with partial last pages."""
    return Workload(name, batch, tuple(seq_lens), n_q_heads, n_kv_heads, block_size, denoise_steps,
                    permille, structure, planted_per_unit)


def _randn_bf16(shape, gen, device):
    return torch.randn(shape, generator=gen, device=device, dtype=torch.float32).to(torch.bfloat16)


def make_inputs(w: Workload, seed: int, device="cpu", spare_pages: int = 0, hostile_tails: bool = False,
                with_block_inputs: bool = True):
    """Draw one set of inputs for workload ``w``.  Returns a dict of torch tensors on ``device``:

      k_pages, v_pages  bf16 [n_pages, page_size, H_kv, d]
      page_table        int32 [batch, max_pages]  (-1 where unused)
      seq_lens          int32 [batch]
      q_rep             bf16 [batch, H_q, d]        representative query (next block)
      q_blk             bf16 [T-1, batch, B, H_q, d]   per-denoise-step block queries
      k_blk, v_blk      bf16 [T-1, batch, B, H_kv, d]  per-step in-block K/V
      planted           list[b][h] -> int64 tensor of planted positions (cpu), or None
    ``hostile_tails`` writes 2^14 into every K slot past seq_len (and into spare pages), so a
    kernel that forgets to mask the tail selects garbage.
    """
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(int(seed))
    cpu_gen = torch.Generator(device="cpu")
    cpu_gen.manual_seed(int(seed) + 7919)

    P, d, Hq, Hkv, G = w.page_size, w.head_dim, w.n_q_heads, w.n_kv_heads, w.group
    pages_per_seq = [(L + P - 1) // P for L in w.seq_lens]
    max_pages = max(pages_per_seq + [1])
    n_used = sum(pages_per_seq)
    n_pages = n_used + spare_pages
    if w.identity_pages:
        perm = torch.arange(n_pages, dtype=torch.int64)
    else:
        perm = torch.randperm(n_pages, generator=cpu_gen)
    page_table = torch.full((w.batch, max_pages), -1, dtype=torch.int32)
    off = 0
    for b, n in enumerate(pages_per_seq):
        page_table[b, :n] = perm[off:off + n].to(torch.int32)
        off += n
    spare = perm[off:]

    q_rep = _randn_bf16((w.batch, Hq, d), gen, dev)
    k_pages = torch.empty((n_pages, P, Hkv, d), dtype=torch.bfloat16, device=dev)
    v_pages = torch.empty((n_pages, P, Hkv, d), dtype=torch.bfloat16, device=dev)
    planted: List[Optional[list]] = []
    page_table_dev = page_table.to(dev)

    for b, L in enumerate(w.seq_lens):
        n = pages_per_seq[b]
        if n == 0:
            planted.append([torch.empty(0, dtype=torch.int64) for _ in range(Hkv)])
            continue
        kb = torch.randn((n * P, Hkv, d), generator=gen, device=dev, dtype=torch.float32)
        vb = torch.randn((n * P, Hkv, d), generator=gen, device=dev, dtype=torch.float32)
        planted_b = []
        if w.structure == "zipf":
            for h in range(Hkv):
                r = torch.randperm(L, generator=cpu_gen).to(dev).to(torch.float32) + 1.0
                kb[:L, h, :] *= (1.0 + 7.0 / r)[:, None]
        if w.structure == "planted" and w.planted_per_unit > 0:
            for h in range(Hkv):
                npl = min(w.planted_per_unit, L)
                pos = torch.randperm(L, generator=cpu_gen)[:npl]
                g_star = (torch.arange(npl) % G) + h * G
                qh = q_rep[b, g_star.to(dev), :].to(torch.float32)
                qh = qh / qh.norm(dim=-1, keepdim=True)
                kb[pos.to(dev), h, :] += 4.0 * qh
                planted_b.append(torch.sort(pos).values)
        else:
            planted_b = [torch.empty(0, dtype=torch.int64) for _ in range(Hkv)]
        planted.append(planted_b)
        if hostile_tails and L < n * P:
            kb[L:, :, :] = 16384.0
        phys = page_table_dev[b, :n].to(torch.int64)
        k_pages[phys] = kb.to(torch.bfloat16).view(n, P, Hkv, d)
        v_pages[phys] = vb.to(torch.bfloat16).view(n, P, Hkv, d)
        del kb, vb
    if spare_pages:
        sp = spare.to(dev)
        k_pages[sp] = 16384.0 if hostile_tails else 0.0
        v_pages[sp] = 0.0

    out = dict(k_pages=k_pages, v_pages=v_pages, page_table=page_table_dev,
               seq_lens=torch.tensor(w.seq_lens, dtype=torch.int32, device=dev).reshape(w.batch),
               q_rep=q_rep, planted=planted)
    if with_block_inputs:
        S = max(w.n_attn_steps, 1)
        out["q_blk"] = _randn_bf16((S, w.batch, w.block_size, Hq, d), gen, dev)
        out["k_blk"] = _randn_bf16((S, w.batch, w.block_size, Hkv, d), gen, dev)
        out["v_blk"] = _randn_bf16((S, w.batch, w.block_size, Hkv, d), gen, dev)
    return out


def to_u16(t: torch.Tensor):
    """bf16 tensor -> host uint16 NumPy array of its bit patterns (what the oracle takes)."""
    import numpy as np
    return t.detach().to("cpu").contiguous().view(torch.int16).numpy().view(np.uint16)


def make_q_x(q_rep: torch.Tensor, x: int, seed: int) -> torch.Tensor:
    """x queries per sequence for the x-query selection sweep (Fig. 8): bf16 [batch, x, H_q, d].
    PAPER.md:145-149: the B queries of a block share one [MASK] embedding and differ only by their position, so
    query 0 is q_rep itself and query j > 0 is q_rep plus a seeded N(0, 1/4) perturbation (the stand-in for the
    RoPE offset of position j; no RoPE is applied anywhere in the synthetic inputs)."""
    batch, Hq, d = q_rep.shape
    gen = torch.Generator(device=q_rep.device)
    gen.manual_seed(int(seed) + 104729)
    noise = torch.randn((batch, x, Hq, d), generator=gen, device=q_rep.device, dtype=torch.float32) * 0.5
    noise[:, 0] = 0.0
    return (q_rep.to(torch.float32)[:, None] + noise).to(torch.bfloat16).contiguous()
