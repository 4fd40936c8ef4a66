"""fp8 (e4m3) KV blocks with per-block power-of-two scales on the GPU against the
oracle: the quantiser bit-exact (codes and scales), the summaries of the fp8 cache bit-exact, whole PRR decode steps
on fp8 pages (scores and block sets bit-exact, outputs within tolerance) and, because the tiles are widened to bf16
exactly on chip, equal BIT FOR BIT to the bf16 path run on the dequantised cache."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import prr_oracle as O
from paper_2606_30389_b200 import prr, synth
import prr_harness as H

pytestmark = pytest.mark.gpu
DEV = "cuda"

TINY = synth.CONFIGS["C0"]
F128 = synth.Config("F128", B=2, L=1, Hq=8, Hkv=2, d=128, ctx_lo=1500, ctx_hi=2040, bs=32, K=8, Bud=12, rho=0.95,
                    steps=6, T_cal=16)
FG7 = synth.Config("FG7", B=1, L=1, Hq=14, Hkv=2, d=128, ctx_lo=4000, ctx_hi=4090, bs=128, K=6, Bud=8, rho=0.7,
                   steps=4, T_cal=16)
SHAPES = [TINY, F128, FG7]


def quantise_on_gpu(cfg, inp):
    MB = inp.block_table.shape[1]
    helper = prr.Context(cfg.Hq, cfg.Hkv, cfg.d, cfg.bs, cfg.K, cfg.Bud, max_batch=cfg.B, max_blocks_per_seq=MB,
                         orchestration=prr.STREAMS)
    kv16 = helper.kv(inp.k_pages, inp.v_pages, inp.block_table, inp.seq_lens)
    k8 = torch.zeros(inp.k_pages.shape, dtype=torch.uint8, device=DEV)
    v8 = torch.zeros_like(k8)
    ks = torch.ones(inp.k_pages.shape[0], cfg.Hkv, dtype=torch.float32, device=DEV)
    vs = torch.ones_like(ks)
    helper.quantize_kv_fp8(kv16, k8, v8, ks, vs)
    torch.cuda.synchronize()
    helper.destroy()
    return k8, v8, ks, vs


def oracle_quantise(cfg, inp):
    table, lens = inp.block_table.cpu().numpy(), inp.seq_lens.cpu().numpy()
    ck, sk = O.quantize_kv_e4m3(synth.bits(inp.k_pages), table, lens, cfg.bs)
    cv, sv = O.quantize_kv_e4m3(synth.bits(inp.v_pages), table, lens, cfg.bs)
    return ck, sk, cv, sv


@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_quantiser_bit_exact(cfg):
    inp = synth.make_layer(cfg, 0, device=DEV, steps=cfg.steps)        # unwritten token slots hold NaN
    k8, v8, ks, vs = quantise_on_gpu(cfg, inp)
    ck, sk, cv, sv = oracle_quantise(cfg, inp)
    assert np.array_equal(k8.cpu().numpy(), ck) and np.array_equal(v8.cpu().numpy(), cv)
    assert np.array_equal(ks.cpu().numpy().view(np.uint32), sk.view(np.uint32))
    assert np.array_equal(vs.cpu().numpy().view(np.uint32), sv.view(np.uint32))
    assert len(np.unique(sk)) > 1                                       # the blocks really have different scales


@pytest.mark.parametrize("policy", [prr.DROP, prr.RETAIN])
@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_decode_steps_on_fp8_pages(cfg, policy):
    inp = synth.make_layer(cfg, 0, device=DEV, steps=cfg.steps)
    k8, v8, ks, vs = quantise_on_gpu(cfg, inp)
    ck, sk, cv, sv = oracle_quantise(cfg, inp)
    dk, dv = O.dequantize_kv_e4m3(ck, sk), O.dequantize_kv_e4m3(cv, sv)  # bf16 bits, exact
    table, lens = inp.block_table.cpu().numpy(), inp.seq_lens.cpu().numpy()
    ol = O.OracleLayer(dk, dv, table, lens, cfg.bs, cfg.K, cfg.Bud, cfg.Hq, policy)
    MB = inp.block_table.shape[1]
    ctx8 = prr.Context(cfg.Hq, cfg.Hkv, cfg.d, cfg.bs, cfg.K, cfg.Bud, max_batch=cfg.B, max_blocks_per_seq=MB,
                       policy=policy, orchestration=prr.STREAMS, kv_dtype=prr.FP8_E4M3)
    out0 = torch.zeros(cfg.B, cfg.Hq, cfg.d, dtype=torch.float32, device=DEV)
    summ0 = torch.zeros(cfg.B, cfg.Hkv, MB, cfg.d, dtype=torch.bfloat16, device=DEV)
    kv8 = ctx8.kv(k8, v8, inp.block_table, inp.seq_lens)
    with pytest.raises(prr.PrrError) as e:                              # scales first
        ctx8.decode_step(kv8, inp.q_dec[0].contiguous(), summ0, out0)
    assert e.value.code == prr.E_STATE
    ctx8.set_kv_scales(0, ks, vs)
    with pytest.raises(prr.PrrError) as e:
        ctx8.append(kv8, inp.k_new[0].contiguous(), inp.v_new[0].contiguous(), summ0)
    assert e.value.code == prr.E_UNSUPPORTED
    gl = H.GpuLayer(cfg, dataclasses.replace(inp, k_pages=k8, v_pages=v8), policy=policy, ctx=ctx8)
    torch.cuda.synchronize()
    assert np.array_equal(synth.bits(gl.summ), ol.summ), "summaries of the fp8 cache"
    # the bf16 path on the dequantised cache: must give the same bits
    to_bf16 = lambda bits: torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).to(DEV)
    twin = H.GpuLayer(cfg, dataclasses.replace(inp, k_pages=to_bf16(dk), v_pages=to_bf16(dv)), policy=policy,
                      orchestration=prr.STREAMS)
    assert torch.equal(twin.summ.view(torch.int16), gl.summ.view(torch.int16))
    gres, ores = gl.calibrate(inp.q_cal), ol.calibrate(synth.bits(inp.q_cal))
    twin.calibrate(inp.q_cal)
    for b in range(cfg.B):
        assert gres[b][0][0] == ores[b][0], "theta*"
    for t in range(cfg.steps):                                          # (no append: see prr_set_kv_scales)
        out = gl.step(t)
        o2 = twin.step(t)
        torch.cuda.synchronize()
        r = ol.step(synth.bits(inp.q_dec[t]))
        sc = gl.scores()
        for b in range(cfg.B):
            nb = ol.n_blocks()[b]
            assert np.array_equal(sc[b, :, :nb].view(np.uint32), r["scores"][b, :, :nb].view(np.uint32)), f"scores t{t}"
        H.compare_sets(gl, r, f"t{t}")
        H.check_out(out.cpu().numpy(), r["out"], f"out t{t}")
        assert torch.equal(out, o2), f"fp8 path vs bf16 path on the dequantised cache, t{t}"
    # partial states of the stage call, fp8 vs bf16-on-dequantised
    P = torch.from_numpy(np.stack([[np.arange(cfg.Bud, dtype=np.int32)] * cfg.Hkv] * cfg.B)).to(DEV)
    q = inp.q_dec[0].contiguous()
    bufs = []
    for g in (gl, twin):
        Op = torch.zeros(cfg.B, cfg.Hq, cfg.Bud, cfg.d, dtype=torch.float32, device=DEV)
        mp = torch.zeros(cfg.B, cfg.Hq, cfg.Bud, dtype=torch.float32, device=DEV)
        lp = torch.zeros_like(mp)
        g.ctx.speculate(g.kv, q, P, Op, mp, lp)
        bufs.append((Op, mp, lp))
    torch.cuda.synchronize()
    for x, y in zip(*bufs):
        assert torch.equal(x, y)
    gl.ctx.check()


def test_fp8_needs_streams_and_small_blocks():
    for kw in (dict(orchestration=prr.FUSED, block_size=64), dict(orchestration=prr.STREAMS, block_size=256)):
        with pytest.raises(prr.PrrError) as e:
            prr.Context(8, 2, 64, kw["block_size"], 8, 8, orchestration=kw["orchestration"], kv_dtype=prr.FP8_E4M3)
        assert e.value.code == prr.E_UNSUPPORTED
