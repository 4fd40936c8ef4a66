"""prr_attend_blocks_static (the entry point that allocates nothing, include/prr.h) against the existing path.

Collected last on purpose (the suite runs with `pytest -x`).  The existing path is prr_repair with an empty
prediction: per-block partial states into ctx-owned buffers, then the Eq. 6-8 fold.  The new entry point runs the
same attention with its partial states in the library's static device array; the two must agree within the
tolerance of the other GPU tests (Q12; in fact to the last bit: same kernels, same fold order), on two
calls in a row that SHARE the array, and both must match the oracle's attention over the block lists.
"""
import numpy as np
import pytest
import torch

from oracle import prr_oracle as O
from paper_2606_30389_b200 import prr, synth
import prr_harness as H

pytestmark = pytest.mark.gpu
DEV = "cuda"

TINY = synth.CONFIGS["C0"]
MID = synth.Config("NA128", B=2, L=1, Hq=8, Hkv=2, d=128, ctx_lo=3000, ctx_hi=4090, bs=64, K=12, Bud=16, rho=0.95,
                   steps=4, T_cal=8)


def random_lists(cfg, nb, rng, holes):
    A = np.full((cfg.B, cfg.Hkv, cfg.K), -1, dtype=np.int32)
    for b in range(cfg.B):
        for h in range(cfg.Hkv):
            k = min(cfg.K, int(nb[b]))
            A[b, h, :k] = np.sort(rng.choice(nb[b], size=k, replace=False))
            if holes:                                   # a hole in the middle of the list is skipped
                A[b, h, (b + h) % k] = -1
    return A


@pytest.mark.parametrize("cfg", [TINY, MID], ids=lambda c: c.name)
def test_static_scratch_attention_matches_existing_path_two_calls(cfg):
    inp = synth.make_layer(cfg, 0, device=DEV, steps=cfg.steps)
    gl = H.GpuLayer(cfg, inp)
    ol = H.oracle_layer(cfg, inp)
    nb = ol.n_blocks()
    rng = np.random.default_rng(11)
    assert prr.lib().prr_static_scratch_bytes() == 8 * 1024 * 1024
    for call in range(2):                               # the second call finds the first call's states in the array
        A = random_lists(cfg, nb, rng, holes=(call == 1))
        Ad = torch.from_numpy(A).to(DEV)
        q = inp.q_dec[call].contiguous()
        out_new = torch.full((cfg.B, cfg.Hq, cfg.d), float("nan"), dtype=torch.float32, device=DEV)
        m_new = torch.zeros(cfg.B, cfg.Hq, dtype=torch.float32, device=DEV)
        l_new = torch.zeros_like(m_new)
        gl.ctx.attend_blocks_static(gl.kv, q, Ad, cfg.K, out_new, m_new, l_new)
        # existing path: compacted ascending lists (prr_repair's contract), empty prediction
        Ac = np.full_like(A, -1)
        for b in range(cfg.B):
            for h in range(cfg.Hkv):
                v = H.unpad(A[b, h])
                Ac[b, h, :len(v)] = v
        out_old = torch.zeros_like(out_new)
        m_old, l_old = torch.zeros_like(m_new), torch.zeros_like(l_new)
        gl.ctx.repair(gl.kv, q, torch.from_numpy(Ac).to(DEV), None, None, None, None, out_old, m_old, l_old)
        torch.cuda.synchronize()
        got, ref = out_new.cpu().numpy(), out_old.cpu().numpy()
        H.check_out(got, ref.astype(np.float64), f"static vs prr_repair, call {call}")
        assert np.array_equal(got, ref), "same kernels, same fold order: the same bits"
        assert torch.equal(m_new, m_old) and torch.equal(l_new, l_old)
        qb = synth.bits(q)
        for b in range(cfg.B):
            S = [H.unpad(A[b, h]) for h in range(cfg.Hkv)]
            want = O.attend(qb[b], ol.k, ol.v, ol.table[b], ol.lens[b], S, cfg.bs)
            H.check_out(got[b], want, f"static vs oracle, call {call} b{b}")
    gl.ctx.check()


def test_static_scratch_rejects_sizes_beyond_the_array():
    cfg = TINY
    inp = synth.make_layer(cfg, 0, device=DEV, steps=1)
    gl = H.GpuLayer(cfg, inp)
    out = torch.zeros(cfg.B, cfg.Hq, cfg.d, dtype=torch.float32, device=DEV)
    q = inp.q_dec[0].contiguous()
    big = torch.full((cfg.B, cfg.Hkv, 1024), -1, dtype=torch.int32, device=DEV)
    n0 = gl.ctx.launch_count()
    with pytest.raises(prr.PrrError) as e:              # width out of range
        gl.ctx.attend_blocks_static(gl.kv, q, big, 1025, out)
    assert e.value.code == prr.E_INVALID
    assert 8 * 64 * 1024 * 130 * 4 > prr.lib().prr_static_scratch_bytes()
    ctx2 = prr.Context(64, 8, 128, 64, 8, 8, max_batch=8, max_blocks_per_seq=64, n_layers=1)
    kv2 = prr.PagedKV(gl.kv.k_pages, gl.kv.v_pages, gl.kv.block_table, gl.kv.seq_lens, 8, 0)
    with pytest.raises(prr.PrrError) as e:
        ctx2.attend_blocks_static(kv2, q, big, 1024, out)
    assert e.value.code == prr.E_UNSUPPORTED and "static scratch" in str(e.value)
    assert gl.ctx.launch_count() == n0 and ctx2.launch_count() == 0
