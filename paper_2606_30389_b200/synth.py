"""Seeded synthetic inputs for the PRR decode hot path.

This module only DRAWS inputs.  It holds none of the method's arithmetic: no
summaries, scores, top-K, EMA or attention.  It is the one module that both the
CUDA path's callers (tests, bench.py) and the oracle's callers (tests) import;
it imports neither of them.

Recipe (BASELINE.json:configs); the paper's own workloads are
real-model traces on public benchmarks that are not available
here, these inputs stand in for their shapes only:

  keys    k_t = N(0, I_d) + g_b * u_b     per (page, KV head): u_b unit vector,
                                          g_b ~ N(0, 0.5^2); rounded to bf16
  values  v_t = N(0, I_d)                 rounded to bf16
  queries q_0 = sqrt(d) * normalize(N(0, I_d)),
          q_t = sqrt(d) * normalize(rho * q_{t-1} + sigma * eps_t), eps_t ~ N(0, I_d)
          independently per query head; sigma = sqrt(1 - rho^2), except the
          literal 0.31 BASELINE.json prints for rho = 0.95; rounded to bf16.
          `warm` drift steps are discarded so step 0 is stationary.
  appends one (k, v) token per sequence per decode step from the key/value recipe,
          with the (u_b, g_b) of the block the token lands in.
  paging  logical block i of sequence b lives in physical page block_table[b, i];
          the table is a seeded random permutation so paging is exercised.
  unwritten token slots are filled with bf16 NaN so that a kernel that forgets
          the `t < seq_len` mask fails loudly.

Everything is a torch tensor on `device`; bf16 tensors are what the CUDA path
reads, and `bits()` gives the same values as uint16 numpy arrays for the oracle.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass

import numpy as np
import torch


@dataclass(frozen=True)
class Config:
    name: str
    B: int            # batch (sequences)
    L: int            # layers (independent seeded caches)
    Hq: int           # query heads
    Hkv: int          # KV heads
    d: int            # head_dim
    ctx_lo: int       # initial context length, tokens (inclusive range)
    ctx_hi: int
    bs: int           # block size, tokens
    K: int            # top-K blocks
    Bud: int          # speculation budget, blocks
    rho: float        # query drift
    steps: int        # decode steps
    seed: int = 0
    T_cal: int = 256  # rows of the synthetic prefill score trajectory

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    @property
    def sigma(self) -> float:
        # BASELINE.json prints 0.31 for rho = 0.95; other rho use sqrt(1-rho^2)
        return 0.31 if self.rho == 0.95 else math.sqrt(1.0 - self.rho * self.rho)

    @property
    def max_blocks(self) -> int:
        return (self.ctx_hi + self.steps + self.bs - 1) // self.bs + 1

    def scaled(self, **kw) -> "Config":
        return dataclasses.replace(self, **kw)


# BASELINE.json:configs, in file order.  C3 prints no budget/rho: 80 and 0.95.
CONFIGS = {
    "C0": Config("C0", B=1, L=1, Hq=8, Hkv=2, d=64, ctx_lo=4096, ctx_hi=4096, bs=64,
                 K=8, Bud=12, rho=0.95, steps=32, T_cal=64),
    "C1": Config("C1", B=1, L=1, Hq=32, Hkv=8, d=128, ctx_lo=32768, ctx_hi=32768, bs=64,
                 K=64, Bud=80, rho=0.95, steps=128),
    "C2": Config("C2", B=1, L=1, Hq=32, Hkv=8, d=128, ctx_lo=131072, ctx_hi=131072, bs=64,
                 K=64, Bud=96, rho=0.95, steps=128),
    "C3": Config("C3", B=16, L=32, Hq=32, Hkv=8, d=128, ctx_lo=16384, ctx_hi=32768, bs=64,
                 K=64, Bud=80, rho=0.95, steps=64),
    "C4": Config("C4", B=4, L=1, Hq=28, Hkv=4, d=128, ctx_lo=131072, ctx_hi=131072, bs=32,
                 K=128, Bud=160, rho=0.7, steps=64),
}


@dataclass
class LayerInputs:
    cfg: Config
    layer: int
    k_pages: torch.Tensor      # bf16 [n_pages, Hkv, bs, d]
    v_pages: torch.Tensor      # bf16 [n_pages, Hkv, bs, d]
    block_table: torch.Tensor  # int32 [B, max_blocks]
    seq_lens: torch.Tensor     # int32 [B]   initial context lengths
    q_cal: torch.Tensor        # bf16 [T_cal, B, Hq, d]  queries of the synthetic prefill trajectory
    q_dec: torch.Tensor        # bf16 [steps, B, Hq, d]
    k_new: torch.Tensor        # bf16 [steps, B, Hkv, d]
    v_new: torch.Tensor        # bf16 [steps, B, Hkv, d]


def _gen(seed: int, layer: int, purpose: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed * 1_000_003 + layer * 1009 + purpose)
    return g


def _unit(x: torch.Tensor) -> torch.Tensor:
    return x / x.norm(dim=-1, keepdim=True)


def _drift(n: int, shape, d: int, rho: float, sigma: float, warm: int, gen, device) -> torch.Tensor:
    """n steps of the query process after `warm` discarded steps -> bf16 [n, *shape, d]."""
    rt = math.sqrt(d)
    q = rt * _unit(torch.randn(*shape, d, generator=gen, device=device, dtype=torch.float32))
    out = torch.empty(n, *shape, d, device=device, dtype=torch.bfloat16)
    for t in range(-warm, n):
        eps = torch.randn(*shape, d, generator=gen, device=device, dtype=torch.float32)
        q = rt * _unit(rho * q + sigma * eps)
        if t >= 0:
            out[t] = q.to(torch.bfloat16)
    return out


def make_layer(cfg: Config, layer: int = 0, device="cpu", steps: int | None = None,
               warm: int = 64, poison: bool = True) -> LayerInputs:
    """All inputs of one layer of `cfg`: initial paged cache, query streams, appended tokens."""
    steps = cfg.steps if steps is None else steps
    B, Hkv, Hq, d, bs = cfg.B, cfg.Hkv, cfg.Hq, cfg.d, cfg.bs
    max_blocks = (cfg.ctx_hi + steps + bs - 1) // bs + 1
    n_pages = B * max_blocks

    g_len = _gen(cfg.seed, layer, 1, "cpu")
    if cfg.ctx_lo == cfg.ctx_hi:
        seq_lens = torch.full((B,), cfg.ctx_lo, dtype=torch.int32)
    else:
        seq_lens = torch.randint(cfg.ctx_lo, cfg.ctx_hi + 1, (B,), generator=g_len, dtype=torch.int32)
    perm = torch.randperm(n_pages, generator=g_len).to(torch.int32).reshape(B, max_blocks)

    g_kv = _gen(cfg.seed, layer, 2, device)
    blk_dir = _unit(torch.randn(n_pages, Hkv, d, generator=g_kv, device=device, dtype=torch.float32))
    blk_gain = 0.5 * torch.randn(n_pages, Hkv, generator=g_kv, device=device, dtype=torch.float32)
    off = (blk_gain[..., None] * blk_dir)[:, :, None, :]                  # [n_pages, Hkv, 1, d]
    k_pages = torch.empty(n_pages, Hkv, bs, d, device=device, dtype=torch.bfloat16)
    v_pages = torch.empty_like(k_pages)
    chunk = max(1, (1 << 24) // (Hkv * bs * d))                           # bound fp32 temporaries
    for p0 in range(0, n_pages, chunk):
        p1 = min(n_pages, p0 + chunk)
        k_pages[p0:p1] = (torch.randn(p1 - p0, Hkv, bs, d, generator=g_kv, device=device,
                                      dtype=torch.float32) + off[p0:p1]).to(torch.bfloat16)
        v_pages[p0:p1] = torch.randn(p1 - p0, Hkv, bs, d, generator=g_kv, device=device,
                                     dtype=torch.float32).to(torch.bfloat16)

    block_table = perm.to(device)
    seq_lens_d = seq_lens.to(device)
    if poison:  # token slots at or beyond seq_len hold NaN until an append writes them
        nan = torch.tensor(float("nan"), dtype=torch.bfloat16, device=device)
        for b in range(B):
            n = int(seq_lens[b])
            first = n // bs
            if n % bs:
                pg = int(perm[b, first])
                k_pages[pg, :, n % bs:, :] = nan
                v_pages[pg, :, n % bs:, :] = nan
                first += 1
            pgs = block_table[b, first:].long()
            k_pages[pgs] = nan
            v_pages[pgs] = nan

    g_q = _gen(cfg.seed, layer, 3, device)
    q_all = _drift(cfg.T_cal + steps, (B, Hq), d, cfg.rho, cfg.sigma, warm, g_q, device)
    q_cal, q_dec = q_all[:cfg.T_cal], q_all[cfg.T_cal:]

    g_a = _gen(cfg.seed, layer, 4, device)
    k_new = torch.empty(steps, B, Hkv, d, device=device, dtype=torch.bfloat16)
    v_new = torch.empty_like(k_new)
    for t in range(steps):
        pos = seq_lens_d.long() + t                                       # [B] slot the token lands in
        pg = block_table[torch.arange(B, device=device), pos // bs].long()
        o = blk_gain[pg][..., None] * blk_dir[pg]                         # [B, Hkv, d]
        k_new[t] = (torch.randn(B, Hkv, d, generator=g_a, device=device, dtype=torch.float32) + o
                    ).to(torch.bfloat16)
        v_new[t] = torch.randn(B, Hkv, d, generator=g_a, device=device, dtype=torch.float32
                               ).to(torch.bfloat16)

    return LayerInputs(cfg, layer, k_pages, v_pages, block_table, seq_lens_d, q_cal, q_dec, k_new, v_new)


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 numpy array of the same bit patterns (what the oracle reads)."""
    assert t.dtype == torch.bfloat16
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def from_bits(a: np.ndarray, device="cpu") -> torch.Tensor:
    """uint16 numpy bit patterns -> bf16 tensor."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).view(torch.bfloat16).to(device)
