"""GPU parity: the CUDA path (through the C-ABI) against the oracle, element by element, on the
same seeded inputs.  Integer / index work is compared bit-exactly; scores bit-exactly; attention
outputs within the tolerance BASELINE.json states (harness.check_out)."""
import numpy as np
import pytest
import torch

from oracle import prr_oracle as O
from paper_2606_30389_b200 import prr, synth
import prr_harness as H

pytestmark = pytest.mark.gpu
DEV = "cuda"

# small shapes that still span several tiles and ragged tails
TINY = synth.CONFIGS["C0"].scaled(ctx_lo=700, ctx_hi=1000, B=3, T_cal=16, steps=8)          # d=64, bs=64, G=4
T128 = synth.Config("T128", B=2, L=1, Hq=14, Hkv=2, d=128, ctx_lo=900, ctx_hi=1300, bs=32, K=8, Bud=11,
                    rho=0.8, steps=8, T_cal=16)                                            # G=7, bs=32
T16 = synth.Config("T16", B=2, L=1, Hq=4, Hkv=4, d=128, ctx_lo=300, ctx_hi=333, bs=16, K=6, Bud=9,
                   rho=0.9, steps=20, T_cal=12)                                            # G=1, bs=16
TB128 = synth.Config("TB128", B=1, L=1, Hq=16, Hkv=1, d=64, ctx_lo=2000, ctx_hi=2000, bs=128, K=5, Bud=7,
                     rho=0.9, steps=6, T_cal=12)                                           # G=16, bs=128
SHAPES = [TINY, T128, T16, TB128]


KERNELS = [prr.KERNEL_PERSISTENT, prr.KERNEL_CLUSTER]   # the two fused kernels (k_step.cu, k_row.cu)
KID = {prr.KERNEL_PERSISTENT: "persistent", prr.KERNEL_CLUSTER: "cluster", None: "auto"}


def make(cfg, policy=prr.DROP, seed=None, budget=None, steps=None, orchestration=prr.FUSED, kernel=None, options=(),
         summary="mean"):
    cfg = cfg if seed is None else cfg.scaled(seed=seed)
    inp = synth.make_layer(cfg, 0, device=DEV, steps=steps)
    gl = H.GpuLayer(cfg, inp, policy=policy, budget=budget, orchestration=orchestration, kernel=kernel, options=options)
    ol = H.oracle_layer(cfg, inp, policy=policy, budget=budget, summary=summary)
    return cfg, inp, gl, ol


@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_summaries_and_append_bit_exact(cfg):
    cfg, inp, gl, ol = make(cfg)
    torch.cuda.synchronize()
    assert np.array_equal(synth.bits(gl.summ), ol.summ)
    for t in range(cfg.steps):
        gl.append(t)
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
    torch.cuda.synchronize()
    assert np.array_equal(gl.seq_lens.cpu().numpy(), ol.lens)
    assert np.array_equal(synth.bits(gl.summ), ol.summ)
    for b in range(cfg.B):
        nb = ol.n_blocks()[b]
        pg = ol.table[b, :nb]
        n_last = ol.lens[b] - (nb - 1) * cfg.bs
        assert np.array_equal(synth.bits(gl.k_pages)[pg[:-1]], ol.k[pg[:-1]])
        assert np.array_equal(synth.bits(gl.v_pages)[pg[-1], :, :n_last], ol.v[pg[-1], :, :n_last])


@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_score_bit_exact(cfg):
    cfg, inp, gl, ol = make(cfg)
    sc = torch.full((cfg.B, cfg.Hkv, gl.MB), 7.0, dtype=torch.float32, device=DEV)
    for t in range(3):
        gl.ctx.score(gl.kv, inp.q_dec[t].contiguous(), gl.summ, sc)
        torch.cuda.synchronize()
        want = ol.scores(synth.bits(inp.q_dec[t]))
        got = sc.cpu().numpy()
        for b in range(cfg.B):
            nb = ol.n_blocks()[b]
            assert np.array_equal(got[b, :, :nb].view(np.uint32), want[b, :, :nb].view(np.uint32))
            assert (got[b, :, nb:] == 7.0).all()          # rows beyond NB are not written


@pytest.mark.parametrize("n,k", [(1, 1), (5, 8), (64, 8), (257, 64), (2048, 64), (4096, 128), (1000, 1000)])
def test_topk_bit_exact_with_ties(n, k):
    rng = np.random.default_rng(n + k)
    Hkv, B, MB = 4, 3, 4100
    ctx = prr.Context(4, Hkv, 64, 64, min(k, 512), 4, max_batch=B, max_blocks_per_seq=MB)
    vals = rng.standard_normal((B, Hkv, MB)).astype(np.float32)
    vals[0] = np.round(vals[0] * 2) / 2                       # heavy ties
    vals[1, :, ::3] = 0.0
    vals[1, :, 1::3] = -0.0                                   # +-0 mix
    vals[2, 0] = 1.25                                         # all equal
    vals[2, 1, : n // 2] = np.inf
    nbs = np.array([n, max(1, n - 3), n], dtype=np.int32)
    idx = torch.full((B, Hkv, k), -7, dtype=torch.int32, device=DEV)
    cnt = torch.zeros(B, Hkv, dtype=torch.int32, device=DEV)
    ctx.topk(torch.from_numpy(vals).to(DEV), torch.from_numpy(nbs).to(DEV), B, k, idx, cnt)
    torch.cuda.synchronize()
    got, gc = idx.cpu().numpy(), cnt.cpu().numpy()
    for b in range(B):
        for h in range(Hkv):
            want = O.topk(vals[b, h, :nbs[b]], k)
            assert gc[b, h] == len(want)
            assert np.array_equal(got[b, h, :len(want)], want), (b, h)
            assert (got[b, h, len(want):] == -1).all()


@pytest.mark.parametrize("cfg", [TINY, T16], ids=lambda c: c.name)
def test_ema_update_predict_bit_exact(cfg):
    cfg, inp, gl, ol = make(cfg)
    rng = np.random.default_rng(3)
    theta = (0.6, 0.3, 0.75)
    gl.ctx.set_ema_params(0, -1, *theta)
    nb0 = ol.n_blocks()
    P = torch.empty(cfg.B, cfg.Hkv, cfg.Bud, dtype=torch.int32, device=DEV)
    Pc = torch.empty(cfg.B, cfg.Hkv, dtype=torch.int32, device=DEV)
    L = torch.empty(cfg.Hkv, gl.MB, dtype=torch.float64, device=DEV)
    V = torch.empty_like(L)
    for step in range(6):
        nb = np.minimum(nb0 - 3 + step, gl.MB).astype(np.int32)   # blocks enter over time
        sc = (rng.standard_normal((cfg.B, cfg.Hkv, gl.MB)) * 0.07).astype(np.float32)
        gl.ctx.predict(0, cfg.B, P, Pc)
        torch.cuda.synchronize()
        for b in range(cfg.B):
            for h in range(cfg.Hkv):
                want = O.ema_predict_set(ol.ema[b][h], theta[2], cfg.Bud)
                assert Pc[b, h].item() == len(want)
                assert np.array_equal(P[b, h, :len(want)].cpu().numpy(), want), (step, b, h)
        gl.ctx.ema_update(0, cfg.B, torch.from_numpy(sc).to(DEV), torch.from_numpy(nb).to(DEV))
        for b in range(cfg.B):
            for h in range(cfg.Hkv):
                O.ema_update(ol.ema[b][h], sc[b, h, :nb[b]], theta[0], theta[1])
        for b in range(cfg.B):
            gl.ctx.get_ema(0, b, L, V)
            torch.cuda.synchronize()
            for h in range(cfg.Hkv):
                n = ol.ema[b][h].n
                assert np.array_equal(L[h, :n].cpu().numpy(), ol.ema[b][h].l[:n])
                assert np.array_equal(V[h, :n].cpu().numpy(), ol.ema[b][h].v[:n])


@pytest.mark.parametrize("cfg", [TINY, T128], ids=lambda c: c.name)
def test_calibrate_matches_oracle(cfg):
    cfg, inp, gl, ol = make(cfg)
    gres = gl.calibrate(inp.q_cal)
    ores = ol.calibrate(synth.bits(inp.q_cal))
    P = torch.empty(cfg.B, cfg.Hkv, cfg.Bud, dtype=torch.int32, device=DEV)
    gl.ctx.predict(0, cfg.B, P)
    torch.cuda.synchronize()
    for b in range(cfg.B):
        (theta, Hs, H_all), traj = gres[b]
        otheta, oH, oH_all, oIS = ores[b]
        assert np.array_equal(traj.cpu().numpy().view(np.uint32), oIS.view(np.uint32))
        assert np.array_equal(np.array(H_all), oH_all), np.abs(np.array(H_all) - oH_all).max()
        assert theta == otheta and Hs == oH
        for h in range(cfg.Hkv):
            want = O.ema_predict_set(ol.ema[b][h], otheta[2], cfg.Bud)
            assert np.array_equal(H.unpad(P[b, h].cpu().numpy()), want)


def test_calibrate_causal_staircase():
    cfg, inp, gl, ol = make(TINY)
    b = 1
    nb = int(ol.n_blocks()[b])
    traj = gl.trajectory(inp.q_cal, b).contiguous()
    nv = np.minimum(np.arange(1, cfg.T_cal + 1) * 2, nb).astype(np.int32)
    theta, Hs, H_all = gl.ctx.calibrate(0, b, traj, n_valid=torch.from_numpy(nv).to(DEV))
    otheta, oH, ostates, oH_all = O.calibrate(traj.cpu().numpy(), cfg.K, cfg.Bud, nv)
    assert np.array_equal(np.array(H_all), oH_all) and theta == otheta
    ns = torch.empty(cfg.Hkv, dtype=torch.int32, device=DEV)
    gl.ctx.get_ema(0, b, n_state=ns)
    torch.cuda.synchronize()
    assert ns.tolist() == [ostates[0].n] * cfg.Hkv


@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_block_partials_against_eq6_8_states(cfg):
    """prr_speculate: per-block (m, l, O) of an arbitrary list incl. the open block and -1 holes."""
    cfg, inp, gl, ol = make(cfg)
    gl.append(0); ol.append(synth.bits(inp.k_new[0]), synth.bits(inp.v_new[0]))   # open block is ragged
    rng = np.random.default_rng(5)
    nb = ol.n_blocks()
    P = np.full((cfg.B, cfg.Hkv, cfg.Bud), -1, dtype=np.int32)
    for b in range(cfg.B):
        for h in range(cfg.Hkv):
            pick = np.sort(rng.choice(nb[b] - 1, size=cfg.Bud - 3, replace=False))
            P[b, h, :cfg.Bud - 3] = pick
            P[b, h, cfg.Bud - 2] = nb[b] - 1                      # after a -1 hole: the open block
    Op = torch.full((cfg.B, cfg.Hq, cfg.Bud, cfg.d), 9.0, dtype=torch.float32, device=DEV)
    mp = torch.full((cfg.B, cfg.Hq, cfg.Bud), 9.0, dtype=torch.float32, device=DEV)
    lp = torch.full((cfg.B, cfg.Hq, cfg.Bud), 9.0, dtype=torch.float32, device=DEV)
    q = inp.q_dec[0].contiguous()
    gl.ctx.speculate(gl.kv, q, torch.from_numpy(P).to(DEV), Op, mp, lp)
    torch.cuda.synchronize()
    Op, mp, lp = Op.cpu().numpy(), mp.cpu().numpy(), lp.cpu().numpy()
    qb = synth.bits(q)
    for b in range(cfg.B):
        for h in range(cfg.Hkv):
            for s in range(cfg.Bud):
                for g in range(cfg.G):
                    hq = h * cfg.G + g
                    if P[b, h, s] < 0:
                        assert (Op[b, hq, s] == 9.0).all() and mp[b, hq, s] == 9.0   # untouched
                        continue
                    st = O.fold(qb[b], ol.k, ol.v, ol.table[b], ol.lens[b],
                                [[P[b, h, s]] if hh == h else [] for hh in range(cfg.Hkv)], cfg.bs)[hq]
                    m, l, On = st
                    assert abs(mp[b, hq, s] - m) <= 1e-5 * max(1.0, abs(m))
                    assert abs(lp[b, hq, s] - l) <= 1e-4 * l
                    H.check_out(Op[b, hq, s] / lp[b, hq, s], On, f"partial b{b} hq{hq} s{s}")


@pytest.mark.parametrize("policy", [prr.DROP, prr.RETAIN])
@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_repair_stage_matches_attention_over_true_set(cfg, policy):
    cfg, inp, gl, ol = make(cfg, policy=policy)
    rng = np.random.default_rng(6)
    nb = ol.n_blocks()
    A = np.full((cfg.B, cfg.Hkv, cfg.K), -1, dtype=np.int32)
    P = np.full((cfg.B, cfg.Hkv, cfg.Bud), -1, dtype=np.int32)
    for b in range(cfg.B):
        for h in range(cfg.Hkv):
            A[b, h] = np.sort(rng.choice(nb[b], size=cfg.K, replace=False))
            npred = [cfg.Bud, 0, cfg.Bud - 2][(b + h) % 3]
            keep = rng.choice(A[b, h], size=min(npred, cfg.K) // 2, replace=False)
            rest = np.setdiff1d(np.arange(nb[b]), A[b, h])
            extra = rng.choice(rest, size=min(len(rest), npred - len(keep)), replace=False) if npred else []
            pp = np.sort(np.concatenate([keep, extra]).astype(np.int32))
            P[b, h, :len(pp)] = pp
    q = inp.q_dec[1].contiguous()
    Op = torch.zeros(cfg.B, cfg.Hq, cfg.Bud, cfg.d, dtype=torch.float32, device=DEV)
    mp = torch.zeros(cfg.B, cfg.Hq, cfg.Bud, dtype=torch.float32, device=DEV)
    lp = torch.zeros_like(mp)
    out = torch.zeros(cfg.B, cfg.Hq, cfg.d, dtype=torch.float32, device=DEV)
    mo = torch.zeros(cfg.B, cfg.Hq, dtype=torch.float32, device=DEV)
    lo = torch.zeros_like(mo)
    Pd, Ad = torch.from_numpy(P).to(DEV), torch.from_numpy(A).to(DEV)
    gl.ctx.speculate(gl.kv, q, Pd, Op, mp, lp)
    gl.ctx.repair(gl.kv, q, Ad, Pd, Op, mp, lp, out, mo, lo)
    torch.cuda.synchronize()
    qb = synth.bits(q)
    for b in range(cfg.B):
        S = [np.union1d(A[b, h], H.unpad(P[b, h])) if policy == prr.RETAIN else A[b, h] for h in range(cfg.Hkv)]
        want = O.attend(qb[b], ol.k, ol.v, ol.table[b], ol.lens[b], S, cfg.bs)
        H.check_out(out[b].cpu().numpy(), want, f"repair b{b}")
        st = O.fold(qb[b], ol.k, ol.v, ol.table[b], ol.lens[b], S, cfg.bs)
        for hq in range(cfg.Hq):
            assert abs(mo[b, hq].item() - st[hq][0]) <= 1e-5 * max(1.0, abs(st[hq][0]))
            assert abs(lo[b, hq].item() - st[hq][1]) <= 1e-4 * st[hq][1]
    _, _, M, cnt = gl.sets()
    for b in range(cfg.B):
        for h in range(cfg.Hkv):
            assert np.array_equal(H.unpad(M[b, h]), np.setdiff1d(A[b, h], P[b, h]))


def run_decode(cfg, policy=prr.DROP, steps=None, calibrate=True, budget=None, seed=None, seq_check=True,
               fused_append=False, orchestration=prr.FUSED, kernel=None, options=(), sequential=False, summary="mean"):
    """Whole decode steps against the oracle: scores and block sets bit-exact, outputs within tolerance, and
    (seq_check) the library's own sequential select-then-attend path within 1e-5 of PRR.  sequential=True
    drives prr_attend itself against the oracle."""
    steps = cfg.steps if steps is None else steps
    cfg, inp, gl, ol = make(cfg, policy=policy, budget=budget, seed=seed, steps=steps, orchestration=orchestration,
                            kernel=kernel, options=options, summary=summary)
    twin = H.GpuLayer(cfg, inp, policy=policy, budget=budget, kernel=kernel, options=options, orchestration=orchestration) if seq_check else None
    if calibrate:
        gres = gl.calibrate(inp.q_cal)
        ores = ol.calibrate(synth.bits(inp.q_cal))
        if twin:
            twin.calibrate(inp.q_cal)
        for b in range(cfg.B):
            assert gres[b][0][0] == ores[b][0], "theta*"
    worst = (0.0, 0.0)
    hits = tot = 0
    for t in range(steps):
        if not fused_append:
            gl.append(t)
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        out = gl.step_append(t, sequential=sequential) if fused_append else gl.step(t, sequential=sequential)
        torch.cuda.synchronize()
        r = ol.step(synth.bits(inp.q_dec[t]))
        if sequential:   # select-then-attend: no speculation, the output is attention over A whatever the policy
            qb = synth.bits(inp.q_dec[t])
            r = dict(r, out=np.stack([O.attend(qb[b], ol.k, ol.v, ol.table[b], ol.lens[b], r["A"][b], cfg.bs)
                                      for b in range(cfg.B)]))
        sc = gl.scores()
        for b in range(cfg.B):
            nb = ol.n_blocks()[b]
            assert np.array_equal(sc[b, :, :nb].view(np.uint32), r["scores"][b, :, :nb].view(np.uint32)), f"scores t{t}"
        if sequential:
            A = gl.sets()[0]
            for b in range(cfg.B):
                for h in range(cfg.Hkv):
                    assert np.array_equal(H.unpad(A[b, h]), r["A"][b][h]), f"t{t} A b{b} h{h}"
        else:
            H.compare_sets(gl, r, f"t{t}")
        e = H.check_out(out.cpu().numpy(), r["out"], f"out t{t}")
        worst = (max(worst[0], e[0]), max(worst[1], e[1]))
        if twin:   # the library's own sequential select-then-attend path
            twin.append(t)
            o2 = twin.step(t, sequential=True)
            torch.cuda.synchronize()
            if policy == prr.DROP:
                assert (out - o2).abs().max().item() <= 1e-5, f"PRR vs sequential t{t}"
        for b in range(cfg.B):
            for h in range(cfg.Hkv):
                hits += len(r["A"][b][h]) - len(r["M"][b][h]); tot += len(r["A"][b][h])
    st = gl.ctx.get_stats()
    if not sequential:
        assert st[0] == tot and st[1] == hits and st[2] == tot - hits
    gl.ctx.check()
    if fused_append and twin:   # the cache, the summaries and the lengths the fused append leaves behind
        assert torch.equal(gl.seq_lens, twin.seq_lens), "seq_lens after fused append"
        assert torch.equal(gl.k_pages.view(torch.int16), twin.k_pages.view(torch.int16)), "k_pages after fused append"
        assert torch.equal(gl.v_pages.view(torch.int16), twin.v_pages.view(torch.int16)), "v_pages after fused append"
        assert torch.equal(gl.summ.view(torch.int16), twin.summ.view(torch.int16)), "summaries after fused append"
    return worst, hits / max(tot, 1)


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
@pytest.mark.parametrize("policy", [prr.DROP, prr.RETAIN])
@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_decode_steps_small_shapes(cfg, policy, kernel):
    run_decode(cfg, policy=policy, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
@pytest.mark.parametrize("policy", [prr.DROP, prr.RETAIN])
@pytest.mark.parametrize("cfg", SHAPES, ids=lambda c: c.name)
def test_step_append_small_shapes(cfg, policy, kernel):
    """prr_step_append (a0 fused into the step's launch) against the oracle and against the
    separate prr_append + prr_attend calls of a twin layer, including the cache it leaves behind."""
    run_decode(cfg, policy=policy, fused_append=True, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
@pytest.mark.parametrize("policy", [prr.DROP, prr.RETAIN])
@pytest.mark.parametrize("cfg", [TINY, T128], ids=lambda c: c.name)
def test_sequential_path_against_oracle(cfg, policy, kernel):
    """prr_attend, the in-library select-then-attend baseline (a10), against the oracle itself: A bit-exact,
    output = attention over A under both policies (nothing is speculated, so nothing is retained)."""
    run_decode(cfg, policy=policy, kernel=kernel, sequential=True, seq_check=False)
    run_decode(cfg, policy=policy, kernel=kernel, sequential=True, seq_check=False, fused_append=True)


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
def test_step_append_block_boundary_and_full_size(kernel):
    """Appends that open a new block (slot 0) and the headline config at full size."""
    run_decode(T16.scaled(ctx_lo=16 * 5, ctx_hi=16 * 5), steps=20, fused_append=True, kernel=kernel)   # starts on a boundary
    run_decode(synth.CONFIGS["C2"].scaled(T_cal=16), steps=4, fused_append=True, kernel=kernel)
    run_decode(synth.CONFIGS["C4"].scaled(T_cal=8), steps=2, fused_append=True, kernel=kernel)


def test_streams_orchestration_whole_steps():
    """PRR_STREAMS: the paper's literal two-stream, event-ordered orchestration of the stage kernels
    (Fig. 1 / Fig. 5), same oracle, same tolerances; prr_step_append falls back to two calls."""
    run_decode(TINY, orchestration=prr.STREAMS)
    run_decode(T128, policy=prr.RETAIN, orchestration=prr.STREAMS, fused_append=True)


def test_timeline_and_check():
    """prr_timeline_*: every warp of the fused step stamps its phase boundaries; prr_check is clean."""
    cfg, inp, gl, ol = make(TINY)
    gl.calibrate(inp.q_cal)
    gl.ctx.timeline_enable(True)
    gl.step_append(0)
    torch.cuda.synchronize()
    tl = gl.ctx.timeline_read().astype(np.int64)
    gl.ctx.timeline_enable(False)
    assert tl.ndim == 2 and tl.shape[1] == 16 and tl.shape[0] >= 148
    live = tl[tl[:, 0] > 0]
    assert len(live) >= 148                                   # one CTA per SM, several warps each
    assert (live[:, 5] >= live[:, 0]).all()                   # merge-done stamp after the start stamp
    assert (live[:, 5] - live[:, 0]).max() < 5_000_000        # a step takes microseconds, not milliseconds
    gl.ctx.check()


def test_decode_c0_full():
    """BASELINE.json configs[0]: every one of the 32 steps, all outputs."""
    worst, hit = run_decode(synth.CONFIGS["C0"])
    assert hit > 0.5


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
def test_decode_without_calibration_and_zero_budget(kernel):
    run_decode(TINY, calibrate=False, kernel=kernel)                 # first step: no state -> P = {} -> repair all of A
    run_decode(TINY, budget=0, seq_check=False, kernel=kernel)       # no speculation at all
    run_decode(T16.scaled(K=40), steps=4, kernel=kernel)             # K > number of blocks


def test_decode_c1_all_steps():
    """BASELINE.json configs[1] at full size (32768 ctx, 512 blocks): all 128 steps, every output compared,
    PRR within 1e-5 of the library's sequential path at every step."""
    run_decode(synth.CONFIGS["C1"].scaled(T_cal=32))
    run_decode(synth.CONFIGS["C1"].scaled(T_cal=32), steps=12, kernel=prr.KERNEL_CLUSTER)


def test_decode_c2_all_steps():
    """configs[2], the headline 128K case, at full size: all 128 steps, every output compared."""
    run_decode(synth.CONFIGS["C2"].scaled(T_cal=16))
    run_decode(synth.CONFIGS["C2"].scaled(T_cal=16), steps=8, kernel=prr.KERNEL_CLUSTER)


def test_decode_c4_all_steps():
    """configs[4]: batch 4, GQA 7, block 32, 4096 blocks, K=128, budget 160, rho 0.7: all 64 steps."""
    run_decode(synth.CONFIGS["C4"].scaled(T_cal=8))
    run_decode(synth.CONFIGS["C4"].scaled(T_cal=8), steps=4, kernel=prr.KERNEL_CLUSTER)


def test_decode_c3_all_layers():
    """configs[3]: batch 16, ragged lengths in [16384, 32768], a stack of 32 independently seeded layers sharing
    ONE context, theta calibrated per (layer, sequence), 8 of the 64 decode steps.  Four layers are resident and
    interleave like a model's forward pass at a time (the oracle's host copy of a layer is 1.6 GB); every layer's
    scores, block sets and outputs are compared at every step, and PRR against the library's own sequential
    path (1e-5) on a twin context."""
    cfg = synth.CONFIGS["C3"].scaled(T_cal=8)
    steps, L, GROUP = 8, cfg.L, 4
    MB = (cfg.ctx_hi + steps + cfg.bs - 1) // cfg.bs + 1
    mk = lambda: prr.Context(cfg.Hq, cfg.Hkv, cfg.d, cfg.bs, cfg.K, cfg.Bud, max_batch=cfg.B, max_blocks_per_seq=MB,
                             n_layers=L)
    ctx, ctx2 = mk(), mk()
    kernels = set()
    for l0 in range(0, L, GROUP):
        layers = []
        for l in range(l0, min(L, l0 + GROUP)):
            inp = synth.make_layer(cfg, l, device=DEV, steps=steps)
            gl = H.GpuLayer(cfg, inp, ctx=ctx, layer=l, n_layers=L)
            twin = H.GpuLayer(cfg, inp, ctx=ctx2, layer=l, n_layers=L)
            ol = H.oracle_layer(cfg, inp)
            gres = gl.calibrate(inp.q_cal)
            twin.calibrate(inp.q_cal)
            ores = ol.calibrate(synth.bits(inp.q_cal))
            for b in range(cfg.B):
                assert gres[b][0][0] == ores[b][0], f"theta* L{l} b{b}"
            layers.append((inp, gl, twin, ol))
        for t in range(steps):
            for inp, gl, twin, ol in layers:          # layers interleave like a model's forward pass
                gl.step_append(t)
                twin.append(t)
                twin.step(t, sequential=True)
            torch.cuda.synchronize()
            kernels.add(ctx.get_option(prr.OPT_LAST_KERNEL))
            for inp, gl, twin, ol in layers:          # every layer keeps its own out buffer
                ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
                r = ol.step(synth.bits(inp.q_dec[t]))
                sc = gl.scores()
                for b in range(cfg.B):
                    nb = ol.n_blocks()[b]
                    assert np.array_equal(sc[b, :, :nb].view(np.uint32), r["scores"][b, :, :nb].view(np.uint32))
                H.compare_sets(gl, r, f"t{t} L{gl.layer}")
                H.check_out(gl.out.cpu().numpy(), r["out"], f"C3 t{t} L{gl.layer}")
                assert (gl.out - twin.out).abs().max().item() <= 1e-5, f"PRR vs sequential t{t} L{gl.layer}"
        del layers
        torch.cuda.empty_cache()
    ctx.check(); ctx2.check()
    assert kernels == {prr.KERNEL_CLUSTER}        # 128 rows: the library runs a cluster per row here


def test_decode_c3_shape_persistent_kernel():
    """The same shape on the other fused kernel: 2 layers, 3 steps."""
    cfg = synth.CONFIGS["C3"].scaled(T_cal=8)
    steps = 3
    MB = (cfg.ctx_hi + steps + cfg.bs - 1) // cfg.bs + 1
    ctx = prr.Context(cfg.Hq, cfg.Hkv, cfg.d, cfg.bs, cfg.K, cfg.Bud, max_batch=cfg.B, max_blocks_per_seq=MB,
                      n_layers=2)
    ctx.set_option(prr.OPT_KERNEL, prr.KERNEL_PERSISTENT)
    layers = []
    for l in range(2):
        inp = synth.make_layer(cfg, l, device=DEV, steps=steps)
        gl = H.GpuLayer(cfg, inp, ctx=ctx, layer=l, n_layers=2)
        ol = H.oracle_layer(cfg, inp)
        gl.ctx.set_ema_params(l, -1, 0.6, 0.2, 0.5)
        ol.theta = [(0.6, 0.2, 0.5)] * cfg.B
        layers.append((inp, gl, ol))
    for t in range(steps):
        for inp, gl, ol in layers:
            gl.append(t)
            gl.step(t)
        torch.cuda.synchronize()
        for inp, gl, ol in layers:
            ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
            r = ol.step(synth.bits(inp.q_dec[t]))
            H.compare_sets(gl, r, f"t{t} L{gl.layer}")
            H.check_out(gl.out.cpu().numpy(), r["out"], f"C3 t{t} L{gl.layer}")


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
@pytest.mark.parametrize("pdl", [1, 0])
@pytest.mark.parametrize("name", ["TINY", "C1", "C2"])
def test_graph_captured_back_to_back_steps(name, pdl, kernel):
    """32 prr_step_append steps captured into ONE graph and replayed without a host synchronisation between
    them (with and without programmatic dependent launch): every out, the final block sets, scores and the
    cache must equal what an eager, step-by-step synchronised twin produces, and the last step the oracle's."""
    cfg = TINY.scaled(steps=32) if name == "TINY" else synth.CONFIGS[name].scaled(T_cal=8)
    n = 32
    cfg, inp, gl, ol = make(cfg, steps=n, kernel=kernel, options=[(prr.OPT_PDL, pdl)])
    _, _, g2, _ = make(cfg, steps=n, kernel=kernel, options=[(prr.OPT_PDL, pdl)])
    gl.calibrate(inp.q_cal); g2.calibrate(inp.q_cal); ol.calibrate(synth.bits(inp.q_cal))
    outs_e = []
    for t in range(n):
        outs_e.append(gl.step_append(t).clone())
        torch.cuda.synchronize()
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = ol.step(synth.bits(inp.q_dec[t]))
    s = torch.cuda.Stream()
    outs_g = [torch.zeros_like(g2.out) for _ in range(n)]
    with torch.cuda.stream(s):
        g2.ctx.graph_begin(s)
        for t in range(n):
            g2.ctx.step_append(g2.kv, inp.q_dec[t].contiguous(), inp.k_new[t].contiguous(), inp.v_new[t].contiguous(),
                               g2.summ, outs_g[t], stream=s)
        graph = g2.ctx.graph_end(s)
        graph.launch(s)
    s.synchronize()
    g2.ctx.check()
    for t in range(n):
        assert (outs_e[t] - outs_g[t]).abs().max().item() <= 2e-6, t
    H.compare_sets(g2, r, "last step of the graph")
    H.check_out(outs_g[-1].cpu().numpy(), r["out"], "last step of the graph")
    assert np.array_equal(g2.scores().view(np.uint32), gl.scores().view(np.uint32))
    assert torch.equal(g2.seq_lens, gl.seq_lens)
    assert torch.equal(g2.k_pages.view(torch.int16), gl.k_pages.view(torch.int16))
    assert torch.equal(g2.summ.view(torch.int16), gl.summ.view(torch.int16))
    graph.destroy()


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
def test_fused_selection_ties(kernel):
    """The fused kernels' own top-K on rows full of ties: keys (hence summaries and scores) of many blocks are
    made identical, a second group is zeroed (score exactly 0), so the K-th and the budget-th rank fall inside
    runs of equal scores and the lower-index rule decides; more than 128 equal candidates at the threshold."""
    cfg = synth.Config("TIES", B=2, L=1, Hq=8, Hkv=2, d=64, ctx_lo=64 * 300, ctx_hi=64 * 300, bs=64, K=40, Bud=60,
                       rho=0.9, steps=4, T_cal=8)
    inp = synth.make_layer(cfg, 0, device=DEV, steps=cfg.steps)
    tab = inp.block_table.long()
    for b in range(cfg.B):
        src = tab[b, 7]
        for i in range(20, 220):          # 200 blocks share one page image: 200 equal scores per row
            inp.k_pages[tab[b, i]] = inp.k_pages[src]
        for i in range(230, 260):         # 30 blocks of zero keys: score +0
            inp.k_pages[tab[b, i]] = 0
    gl = H.GpuLayer(cfg, inp, kernel=kernel)
    ol = H.oracle_layer(cfg, inp)
    gl.ctx.set_ema_params(0, -1, 0.8, 0.1, 0.25)
    ol.theta = [(0.8, 0.1, 0.25)] * cfg.B
    for t in range(cfg.steps):
        out = gl.step_append(t)
        torch.cuda.synchronize()
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = ol.step(synth.bits(inp.q_dec[t]))
        H.compare_sets(gl, r, f"ties t{t}")
        H.check_out(out.cpu().numpy(), r["out"], f"ties t{t}")
    gl.ctx.check()


def test_streams_orchestration_full_size_and_graph():
    """PRR_STREAMS (the paper's literal two-stream, event-ordered orchestration) at configs[1] size, and captured
    into a graph: several steps without a host synchronisation, starting one token before a block boundary so
    the append of the next step crosses it while the EMA update of the previous one may still be running."""
    run_decode(synth.CONFIGS["C1"].scaled(T_cal=8), steps=4, orchestration=prr.STREAMS)
    cfg = T16.scaled(ctx_lo=16 * 6 - 1, ctx_hi=16 * 6 - 1, steps=12)
    cfg, inp, gl, ol = make(cfg, orchestration=prr.STREAMS)
    _, _, g2, _ = make(cfg, orchestration=prr.STREAMS)
    for g in (gl, g2):
        g.ctx.set_ema_params(0, -1, 0.6, 0.2, 0.5)
    ol.theta = [(0.6, 0.2, 0.5)] * cfg.B
    n = cfg.steps
    for t in range(n):                                  # no host synchronisation between the steps
        gl.append(t); gl.step(t)
    torch.cuda.synchronize()
    for t in range(n):
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = ol.step(synth.bits(inp.q_dec[t]))
    H.compare_sets(gl, r, "streams, unsynchronised steps")
    H.check_out(gl.out.cpu().numpy(), r["out"], "streams, unsynchronised steps")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        g2.ctx.graph_begin(s)
        for t in range(n):
            g2.ctx.append(g2.kv, inp.k_new[t].contiguous(), inp.v_new[t].contiguous(), g2.summ, stream=s)
            g2.ctx.decode_step(g2.kv, inp.q_dec[t].contiguous(), g2.summ, g2.out, stream=s)
        graph = g2.ctx.graph_end(s)
        graph.launch(s)
    s.synchronize()
    H.compare_sets(g2, r, "streams in a graph")
    H.check_out(g2.out.cpu().numpy(), r["out"], "streams in a graph")
    graph.destroy()


@pytest.mark.parametrize("kernel", KERNELS, ids=KID.get)
@pytest.mark.parametrize("cfg", [TINY, T128], ids=lambda c: c.name)
def test_runtime_budget_varies_per_step(cfg, kernel):
    """prr_set_budget (delta is a run-time choice): the budget changes between steps, down to
    0 (no speculation) and back to the maximum; A, P, M stay bit-exact against the oracle run with the same
    per-step budget, outputs in tolerance, PRR within 1e-5 of the sequential path."""
    cfg, inp, gl, ol = make(cfg, kernel=kernel, steps=8)
    twin = H.GpuLayer(cfg, inp, kernel=kernel)
    gl.calibrate(inp.q_cal); twin.calibrate(inp.q_cal); ol.calibrate(synth.bits(inp.q_cal))
    plan = [cfg.Bud, cfg.K, 3, 0, 0, cfg.Bud, 1, cfg.K // 2]
    for t in range(8):
        gl.ctx.set_budget(0, plan[t]); ol.budget = plan[t]
        assert gl.ctx.get_budget(0) == plan[t]
        out = gl.step_append(t)
        twin.append(t); o2 = twin.step(t, sequential=True)
        torch.cuda.synchronize()
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = ol.step(synth.bits(inp.q_dec[t]))
        for b in range(cfg.B):
            for h in range(cfg.Hkv):
                assert len(r["P"][b][h]) <= plan[t]
        H.compare_sets(gl, r, f"budget {plan[t]} t{t}")
        H.check_out(out.cpu().numpy(), r["out"], f"budget {plan[t]} t{t}")
        assert (out - o2).abs().max().item() <= 1e-5
    with pytest.raises(prr.PrrError):
        gl.ctx.set_budget(0, cfg.Bud + 1)


@pytest.mark.parametrize("mode", ["k_step", "k_row", "streams"])
def test_per_sequence_budgets_in_one_batch(mode):
    """prr_set_budget_seq: the sequences of ONE batch carry different run-time budgets (one of
    them 0 = no speculation, one the layer's), changed between steps; A, P, M bit-exact against the oracle run with
    the same per-sequence budgets, outputs in tolerance, PRR within 1e-5 of the sequential path."""
    cfg = TINY                                                   # B = 3
    kw = dict(kernel={"k_step": 1, "k_row": 2}.get(mode)) if mode != "streams" else dict(orchestration=prr.STREAMS)
    cfg, inp, gl, ol = make(cfg, steps=8, **kw)
    twin = H.GpuLayer(cfg, inp, **kw)
    gl.calibrate(inp.q_cal); twin.calibrate(inp.q_cal); ol.calibrate(synth.bits(inp.q_cal))
    plans = [[0, None, 5], [0, None, 5], [cfg.Bud, 0, None], [3, 0, None], [None, None, None], [0, 0, 0], [1, cfg.K, 0],
             [None, 2, cfg.Bud]]
    for t in range(8):
        for b in range(cfg.B):
            v = plans[t][b]
            gl.ctx.set_budget_seq(0, b, -1 if v is None else v)
            assert gl.ctx.get_budget_seq(0, b) == (cfg.Bud if v is None else v)
        ol.budget_seq = plans[t]
        out = gl.step_append(t) if mode != "streams" else (gl.append(t), gl.step(t))[1]
        twin.append(t); o2 = twin.step(t, sequential=True)
        torch.cuda.synchronize()
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = ol.step(synth.bits(inp.q_dec[t]))
        for b in range(cfg.B):
            cap = cfg.Bud if plans[t][b] is None else plans[t][b]
            assert all(len(r["P"][b][h]) <= cap for h in range(cfg.Hkv))
        H.compare_sets(gl, r, f"per-seq budgets {plans[t]} t{t}")
        H.check_out(out.cpu().numpy(), r["out"], f"per-seq budgets t{t}")
        assert (out - o2).abs().max().item() <= 1e-5
    with pytest.raises(prr.PrrError):
        gl.ctx.set_budget_seq(0, cfg.B, 1)                       # seq out of range
    with pytest.raises(prr.PrrError):
        gl.ctx.set_budget_seq(0, 0, cfg.Bud + 1)
    gl.ctx.check()


def test_profile_budget_leaves_no_trace_and_fit():
    """prr_profile_budget sweeps candidate budgets on the layer's cache (section 4.4 in the library) and
    restores the predictor state: the decode steps after it still match the oracle bit-exactly.  prr_budget_fit /
    prr_budget_for: a polynomial through profiled points, pinned on exactly representable data."""
    cfg, inp, gl, ol = make(TINY, steps=6)
    gl.calibrate(inp.q_cal); ol.calibrate(synth.bits(inp.q_cal))
    for t in range(2):
        gl.step_append(t); ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t])); r = ol.step(synth.bits(inp.q_dec[t]))
    cands = [0, 4, cfg.K, cfg.Bud]
    us, seq_us, best = gl.ctx.profile_budget(gl.kv, inp.q_cal.contiguous(), gl.summ, cands, cold_l2=False)
    assert len(us) == 4 and all(0.5 < u < 5000 for u in us) and 0.5 < seq_us < 5000
    assert best in cands
    assert gl.ctx.get_budget(0) == cfg.Bud
    for t in range(2, 6):
        out = gl.step_append(t)
        torch.cuda.synchronize()
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t])); r = ol.step(synth.bits(inp.q_dec[t]))
        H.compare_sets(gl, r, f"after profiling t{t}")
        H.check_out(out.cpu().numpy(), r["out"], f"after profiling t{t}")
    c = gl.ctx
    assert c.budget_for(12345) == cfg.Bud                          # nothing fitted yet: the budget of prr_create
    c.budget_fit([4096, 8192, 16384, 32768], [12, 10, 6, 2], degree=3)   # 4 points, degree 3: interpolation
    assert [c.budget_for(x) for x in (4096, 8192, 16384, 32768)] == [12, 10, 6, 2]
    c.budget_fit([1000, 2000, 3000], [3, 5, 7], degree=1)                # exactly linear data
    assert [c.budget_for(x) for x in (1000, 1500, 2000, 2500, 3000)] == [3, 4, 5, 6, 7]
    assert c.budget_for(0) == 1 and c.budget_for(10 ** 6) == cfg.Bud     # clamped to [0, budget of prr_create]
    c.budget_fit([5000], [9], degree=2)                                  # one point: a constant
    assert c.budget_for(1) == 9 and c.budget_for(99999) == 9


@pytest.mark.parametrize("mode,kernel", [(prr.MODE_S2, prr.KERNEL_PERSISTENT), (prr.MODE_S2, prr.KERNEL_CLUSTER),
                                         (prr.MODE_S1, None), (prr.MODE_S3, None)], ids=["S2-persistent", "S2-cluster", "S1", "S3"])
@pytest.mark.parametrize("cfg", [TINY, T128], ids=lambda c: c.name)
def test_ablation_modes(cfg, mode, kernel):
    """S1 = reuse the last top-K and recompute on any miss, S2 = reuse + repair, S3 = EMA + repair.
    S1 / S2 predict P_t = A_{t-1} (the oracle with theta = (1, 1, 0), budget K: pinned in test_oracle_pins); the
    output is attention over A in every mode, the modes differ in the work done."""
    cfg, inp, gl, ol = make(cfg, kernel=kernel)
    if mode == prr.MODE_S3:
        gl.calibrate(inp.q_cal); ol.calibrate(synth.bits(inp.q_cal))
    gl.ctx.set_mode(mode)
    if mode != prr.MODE_S3:
        ol.theta = [(1.0, 1.0, 0.0)] * cfg.B
        ol.budget = min(cfg.K, cfg.Bud)
    prevA = None
    for t in range(cfg.steps):
        out = gl.step_append(t)
        torch.cuda.synchronize()
        ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = ol.step(synth.bits(inp.q_dec[t]))
        A, P, M = H.compare_sets(gl, r, f"mode {mode} t{t}")
        if mode != prr.MODE_S3 and prevA is not None:
            assert np.array_equal(P[..., :cfg.K], prevA)               # the prediction IS the last true set
        prevA = A
        H.check_out(out.cpu().numpy(), r["out"], f"mode {mode} t{t}")
    if mode == prr.MODE_S1:
        assert gl.ctx.get_option(prr.OPT_LAST_KERNEL) == prr.KERNEL_CLUSTER
    gl.ctx.check()


def test_block_size_256():
    """Table 3 of the paper sweeps block sizes 16 .. 256: a 256-token block is four sub-tiles of the
    cluster kernel; whole steps against the oracle, open block ragged."""
    cfg = synth.Config("T256", B=2, L=1, Hq=8, Hkv=2, d=128, ctx_lo=256 * 9 + 5, ctx_hi=256 * 12 + 201, bs=256, K=3, Bud=5,
                       rho=0.9, steps=6, T_cal=8)
    run_decode(cfg, fused_append=True)
    run_decode(cfg, policy=prr.RETAIN)
    with pytest.raises(prr.PrrError) as e:
        prr.Context(8, 2, 128, 256, 3, 5, orchestration=prr.STREAMS)
    assert e.value.code == prr.E_UNSUPPORTED


def test_graph_replay_matches_eager():
    cfg, inp, gl, ol = make(TINY)
    _, _, g2, _ = make(TINY)
    gl.calibrate(inp.q_cal); g2.calibrate(inp.q_cal)
    outs_e = []
    for t in range(4):
        gl.append(t); outs_e.append(gl.step(t).clone())
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    outs_g = [torch.zeros_like(g2.out) for _ in range(4)]
    with torch.cuda.stream(s):
        g2.ctx.graph_begin(s)
        for t in range(4):
            g2.ctx.append(g2.kv, inp.k_new[t].contiguous(), inp.v_new[t].contiguous(), g2.summ, stream=s)
            g2.ctx.decode_step(g2.kv, inp.q_dec[t].contiguous(), g2.summ, outs_g[t], stream=s)
        graph = g2.ctx.graph_end(s)
        graph.launch(s)
    s.synchronize()
    for t in range(4):   # (the fold order of the partial states follows the tile arrival order: equal to fp32 rounding, not bitwise)
        assert (outs_e[t] - outs_g[t]).abs().max().item() <= 2e-6, t
    assert g2.seq_lens.tolist() == gl.seq_lens.tolist()
    graph.destroy()


def test_host_buffer_step_matches_device_step():
    cfg, inp, gl, ol = make(TINY)
    _, _, g2, _ = make(TINY)
    out_h = torch.zeros(cfg.B, cfg.Hq, cfg.d, dtype=torch.float32).pin_memory()
    for t in range(3):
        gl.append(t); o = gl.step(t)
        g2.ctx.decode_step_host(g2.kv, inp.q_dec[t].cpu().contiguous().pin_memory(),
                                inp.k_new[t].cpu().contiguous().pin_memory(),
                                inp.v_new[t].cpu().contiguous().pin_memory(), g2.summ, out_h)
        torch.cuda.synchronize()
        assert (o.cpu() - out_h).abs().max().item() <= 2e-6


def test_errors_are_reported_not_raised_in_c():
    with pytest.raises(prr.PrrError) as e:
        prr.Context(30, 8, 128, 64, 8, 8)
    assert e.value.code == prr.E_INVALID
    with pytest.raises(prr.PrrError) as e:
        prr.Context(32, 8, 96, 64, 8, 8)
    assert e.value.code == prr.E_UNSUPPORTED
    cfg, inp, gl, ol = make(TINY)
    with pytest.raises(prr.PrrError) as e:
        gl.ctx.score(gl.kv, None, gl.summ, gl.out)
    assert e.value.code == prr.E_INVALID and "null" in str(e.value)
    bad = gl.ctx.kv(gl.k_pages, gl.v_pages, inp.block_table, gl.seq_lens, layer=3)
    with pytest.raises(prr.PrrError):
        gl.ctx.decode_step(bad, inp.q_dec[0].contiguous(), gl.summ, gl.out)


def test_quest_minmax_summaries():
    """§8(f)-2: Quest's channel-wise min / max block metadata scored with the GQA mean query (A.1).
    Summaries (bulk and after appends) and scores bit-exact against the oracle; whole decode steps (both policies,
    PRR and select-then-attend) run on them under PRR_STREAMS; a PRR_FUSED context refuses the option."""
    q_opt = ((prr.OPT_SUMMARY, prr.SUMMARY_QUEST),)
    for cfg in (TINY, T16, synth.CONFIGS["C1"].scaled(T_cal=8, steps=3)):
        cfg, inp, gl, ol = make(cfg, orchestration=prr.STREAMS, options=q_opt, summary="quest")
        torch.cuda.synchronize()
        assert gl.summ.shape[-2:] == (2, cfg.d)
        assert np.array_equal(synth.bits(gl.summ), ol.summ), "bulk min / max"
        for t in range(cfg.steps):
            gl.append(t)
            ol.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        torch.cuda.synchronize()
        assert np.array_equal(synth.bits(gl.summ), ol.summ), "min / max after appends"
        assert np.array_equal(gl.seq_lens.cpu().numpy(), ol.lens)
    run_decode(TINY, orchestration=prr.STREAMS, options=q_opt, summary="quest")
    run_decode(T128, policy=prr.RETAIN, orchestration=prr.STREAMS, options=q_opt, summary="quest", fused_append=True)
    run_decode(T16, orchestration=prr.STREAMS, options=q_opt, summary="quest", sequential=True, seq_check=False)
    run_decode(synth.CONFIGS["C2"].scaled(T_cal=8), steps=3, orchestration=prr.STREAMS, options=q_opt, summary="quest")
    ctx = prr.Context(8, 2, 64, 16, 4, 4, max_batch=1, max_blocks_per_seq=32)
    with pytest.raises(prr.PrrError):
        ctx.set_option(prr.OPT_SUMMARY, prr.SUMMARY_QUEST)
