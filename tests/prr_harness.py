"""Side-by-side drivers for the parity tests: the CUDA path (through the C-ABI binding) and the
oracle run on the same seeded inputs.  Nothing here computes any of the method's arithmetic."""
from __future__ import annotations

import numpy as np
import torch

from oracle import prr_oracle as O
from paper_2606_30389_b200 import prr, synth

ABS_TOL = 2e-3   # BASELINE.json north_star: max-abs 2e-3, max-rel 1e-2 (bf16 in, fp32 accumulate)
REL_TOL = 1e-2


def check_out(got: np.ndarray, want: np.ndarray, what=""):
    """max|x-y| <= 2e-3 and, per (seq, head) vector, ||x-y||inf <= 1e-2 ||y||inf (Q12)."""
    got = np.asarray(got, dtype=np.float64)
    err = np.abs(got - want)
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    assert err.max() <= ABS_TOL, f"{what}: max-abs {err.max():.3e}"
    rel = err.max(axis=-1) / np.maximum(np.abs(want).max(axis=-1), 1e-30)
    assert rel.max() <= REL_TOL, f"{what}: max-rel {rel.max():.3e}"
    return float(err.max()), float(rel.max())


class GpuLayer:
    """One layer of a config on the GPU: owns the caller-side buffers of include/prr.h."""

    def __init__(self, cfg: synth.Config, inp: synth.LayerInputs, policy=prr.DROP, ctx=None, layer=0,
                 n_layers=1, budget=None, orchestration=prr.FUSED, kernel=None, options=()):
        self.cfg, self.inp, self.layer = cfg, inp, layer
        dev = inp.k_pages.device
        self.MB = inp.block_table.shape[1]
        self.Bud = cfg.Bud if budget is None else budget
        self.ctx = ctx or prr.Context(cfg.Hq, cfg.Hkv, cfg.d, cfg.bs, cfg.K, self.Bud, max_batch=cfg.B,
                                      max_blocks_per_seq=self.MB, n_layers=n_layers, policy=policy,
                                      orchestration=orchestration)
        if kernel is not None:
            self.ctx.set_option(prr.OPT_KERNEL, kernel)
        for opt, val in options:
            self.ctx.set_option(opt, val)
        self.k_pages, self.v_pages = inp.k_pages.clone(), inp.v_pages.clone()
        self.seq_lens = inp.seq_lens.clone()
        self.kv = self.ctx.kv(self.k_pages, self.v_pages, inp.block_table, self.seq_lens, layer)
        quest = self.ctx.get_option(prr.OPT_SUMMARY) == prr.SUMMARY_QUEST      # rows hold min then max: 2 d
        self.summ = torch.zeros((cfg.B, cfg.Hkv, self.MB) + ((2, cfg.d) if quest else (cfg.d,)), dtype=torch.bfloat16, device=dev)
        self.out = torch.zeros(cfg.B, cfg.Hq, cfg.d, dtype=torch.float32, device=dev)
        self.ctx.build_summaries(self.kv, self.summ)

    def n_blocks(self):
        return (self.seq_lens.cpu().numpy().astype(np.int64) + self.cfg.bs - 1) // self.cfg.bs

    def trajectory(self, q_cal, b):
        """fp32 [Hkv, T, N_b] prefill score trajectory of sequence b, scored by prr_score."""
        cfg = self.cfg
        nb = int(self.n_blocks()[b])
        T = q_cal.shape[0]
        sc = torch.zeros(cfg.B, cfg.Hkv, self.MB, dtype=torch.float32, device=q_cal.device)
        traj = torch.empty(cfg.Hkv, T, nb, dtype=torch.float32, device=q_cal.device)
        for t in range(T):
            self.ctx.score(self.kv, q_cal[t].contiguous(), self.summ, sc)
            traj[:, t, :] = sc[b, :, :nb]
        return traj

    def calibrate(self, q_cal):
        res = []
        for b in range(self.cfg.B):
            traj = self.trajectory(q_cal, b).contiguous()
            res.append((self.ctx.calibrate(self.layer, b, traj), traj))
        return res

    def append(self, t):
        self.ctx.append(self.kv, self.inp.k_new[t].contiguous(), self.inp.v_new[t].contiguous(), self.summ)

    def step(self, t, sequential=False):
        q = self.inp.q_dec[t].contiguous()
        (self.ctx.attend if sequential else self.ctx.decode_step)(self.kv, q, self.summ, self.out)
        return self.out

    def step_append(self, t, sequential=False):
        """prr_step_append: a0-a8 in one call (one launch with the fused orchestration)."""
        self.ctx.step_append(self.kv, self.inp.q_dec[t].contiguous(), self.inp.k_new[t].contiguous(),
                             self.inp.v_new[t].contiguous(), self.summ, self.out, sequential=sequential)
        return self.out

    def sets(self):
        cfg = self.cfg
        dev = self.out.device
        A = torch.empty(cfg.B, cfg.Hkv, cfg.K, dtype=torch.int32, device=dev)
        P = torch.full((cfg.B, cfg.Hkv, max(self.Bud, 1)), -1, dtype=torch.int32, device=dev)
        M = torch.empty(cfg.B, cfg.Hkv, cfg.K, dtype=torch.int32, device=dev)
        cnt = torch.empty(cfg.B, cfg.Hkv, 3, dtype=torch.int32, device=dev)
        self.ctx.get_sets(self.layer, cfg.B, A, P if self.Bud else None, M, cnt)
        torch.cuda.synchronize()
        return A.cpu().numpy(), P.cpu().numpy()[..., :self.Bud], M.cpu().numpy(), cnt.cpu().numpy()

    def scores(self):
        sc = torch.empty(self.cfg.B, self.cfg.Hkv, self.MB, dtype=torch.float32, device=self.out.device)
        self.ctx.get_scores(self.layer, self.cfg.B, sc)
        torch.cuda.synchronize()
        return sc.cpu().numpy()


def oracle_layer(cfg, inp, policy=O.DROP, budget=None, summary="mean") -> O.OracleLayer:
    return O.OracleLayer(synth.bits(inp.k_pages), synth.bits(inp.v_pages), inp.block_table.cpu().numpy(),
                         inp.seq_lens.cpu().numpy(), cfg.bs, cfg.K, cfg.Bud if budget is None else budget,
                         cfg.Hq, policy, summary)


def unpad(row):
    row = np.asarray(row)
    return row[row >= 0]


def compare_sets(gl: GpuLayer, r: dict, what=""):
    """Bit-exact A, P, M against the oracle's step result."""
    A, P, M, cnt = gl.sets()
    for b in range(gl.cfg.B):
        for h in range(gl.cfg.Hkv):
            assert np.array_equal(unpad(A[b, h]), r["A"][b][h]), f"{what} A b{b} h{h}"
            assert np.array_equal(unpad(P[b, h]), r["P"][b][h]), f"{what} P b{b} h{h}"
            assert np.array_equal(unpad(M[b, h]), r["M"][b][h]), f"{what} M b{b} h{h}"
            assert cnt[b, h].tolist() == [len(r["A"][b][h]), len(r["P"][b][h]), len(r["M"][b][h])]
    return A, P, M
