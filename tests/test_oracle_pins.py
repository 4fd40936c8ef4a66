"""Pins for oracle/prr_oracle.py against things other than itself: exact rational arithmetic,
brute force, closed forms, library routines (torch SDPA, torch bf16 rounding), invariants and the
constants the paper prints (tests/golden/).  CPU only."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

from oracle import prr_oracle as O
from paper_2606_30389_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rand_bf16(rng, shape, scale=1.0):
    x = (rng.standard_normal(shape) * scale).astype(np.float32)
    return synth.bits(torch.from_numpy(x).to(torch.bfloat16))


def frac_of_bf16(b):
    """bf16 bit pattern -> exact Fraction, decoded field by field (independent of the oracle)."""
    b = int(b)
    s = -1 if b >> 15 else 1
    e = (b >> 7) & 0xFF
    m = b & 0x7F
    if e == 0:
        return s * Fraction(m, 1 << 7) * Fraction(1, 1 << 126)
    return s * (1 + Fraction(m, 1 << 7)) * (Fraction(2) ** (e - 127))


def nearest_f32(fr: Fraction) -> np.float32:
    """Correctly rounded float32 of an exact rational (via an exact float64 neighbour search)."""
    x = np.float32(float(fr))
    best = None
    for c in (np.nextafter(x, np.float32(-np.inf)), x, np.nextafter(x, np.float32(np.inf))):
        err = abs(Fraction(float(c)) - fr)
        even = (int(np.float32(c).view(np.uint32)) & 1) == 0
        key = (err, 0 if even else 1)
        if best is None or key < best[0]:
            best = (key, c)
    return np.float32(best[1])


# ------------------------------------------------------------------------------- bf16 rounding
def test_bf16_widen_roundtrip_all_patterns():
    bits = np.arange(0x0080, 0x7F80, dtype=np.uint16)            # positive normals
    bits = np.concatenate([bits, bits | np.uint16(0x8000)])
    x = O.bf16_to_f64(bits)
    assert [frac_of_bf16(b) for b in bits[::997]] == [Fraction(float(v)) for v in x[::997]]
    assert np.array_equal(O.f64_to_bf16(x), bits)


def test_bf16_rne_matches_torch_on_fp32_values():
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(200000) * np.exp(rng.uniform(-20, 20, 200000))).astype(np.float32)
    want = synth.bits(torch.from_numpy(x).to(torch.bfloat16))     # library RNE from fp32
    got = O.f64_to_bf16(x.astype(np.float64))
    assert np.array_equal(got, want)


def test_bf16_rne_ties_and_fp64_only_information():
    one = 1.0
    ulp = 2.0 ** -7
    # exact midpoints go to the even significand
    assert O.f64_to_bf16(np.array([one + ulp / 2]))[0] == 0x3F80          # 1.0 (even)
    assert O.f64_to_bf16(np.array([one + ulp + ulp / 2]))[0] == 0x3F82    # 1+2ulp (even)
    # a hair above the midpoint, visible only in fp64, must round up (no double rounding via fp32)
    assert O.f64_to_bf16(np.array([one + ulp / 2 + 2.0 ** -50]))[0] == 0x3F81
    assert O.f64_to_bf16(np.array([-(one + ulp / 2 + 2.0 ** -50)]))[0] == 0xBF81
    assert O.f64_to_bf16(np.array([0.0]))[0] == 0


# ------------------------------------------------------------------------------------- summary
def _tiny_cache(rng, B=2, Hkv=2, d=8, bs=4, lens=(9, 6), extra=1, scale=1.0):
    mb = max((n + bs - 1) // bs for n in lens) + extra
    n_pages = B * mb
    k = rand_bf16(rng, (n_pages, Hkv, bs, d), scale)
    v = rand_bf16(rng, (n_pages, Hkv, bs, d))
    table = rng.permutation(n_pages).astype(np.int32).reshape(B, mb)
    return k, v, table, np.array(lens, dtype=np.int64), bs


def test_summary_bruteforce_exact_rational():
    rng = np.random.default_rng(2)
    k, v, table, lens, bs = _tiny_cache(rng)
    got = O.summarize(k, table, lens, bs)
    for b in range(2):
        nb = (lens[b] + bs - 1) // bs
        for h in range(2):
            for i in range(nb):
                n_i = min(bs, lens[b] - i * bs)
                for j in range(8):
                    mean = sum(frac_of_bf16(k[table[b, i], h, t, j]) for t in range(n_i)) / n_i
                    # nearest bf16 by exhaustive search over the 3 neighbours of the float guess
                    g = int(got[b, h, i, j])
                    cands = [g - 1, g, g + 1]
                    errs = [abs(frac_of_bf16(c) - mean) for c in cands]
                    assert errs[1] == min(errs), (b, h, i, j)
                    if errs[1] in (errs[0], errs[2]) and mean != frac_of_bf16(g):
                        assert g % 2 == 0                         # tie -> even
    assert not got[0, :, 3:].any() and not got[1, :, 2:].any()    # beyond NB untouched (zero)


def test_summary_identical_keys_and_power_of_two():
    rng = np.random.default_rng(3)
    k, v, table, lens, bs = _tiny_cache(rng, lens=(8, 8))
    row = k[table[0, 1], 1, 0].copy()
    k[table[0, 1], 1, :, :] = row
    got = O.summarize(k, table, lens, bs)
    assert np.array_equal(got[0, 1, 1], row)
    # block of 4 small integers: mean exact, representable
    k[table[1, 0], 0, :, 0] = synth.bits(torch.tensor([1.0, 2.0, 3.0, 6.0]).to(torch.bfloat16))
    got = O.summarize(k, table, lens, bs)
    assert O.bf16_to_f64(got[1, 0, 0, 0]) == 3.0


# --------------------------------------------------------------------------------------- score
def test_score_exact_rational_d64_g4():
    """c = 1/(4*sqrt(64)) = 1/32 is exact, so the oracle must return the correctly rounded fp32
    of the exact rational (sum_g sum_j q*kbar)/32."""
    rng = np.random.default_rng(4)
    B, Hkv, G, d, nb = 2, 2, 4, 64, 5
    q = rand_bf16(rng, (B, Hkv * G, d), 8.0)
    kb = rand_bf16(rng, (B, Hkv, nb + 2, d), 0.2)
    got = O.score(q, kb, np.array([nb, nb - 1]))
    for b in range(B):
        for h in range(Hkv):
            for i in range(nb - b):
                ex = sum(frac_of_bf16(q[b, h * G + g, j]) * frac_of_bf16(kb[b, h, i, j])
                         for g in range(G) for j in range(d)) / 32
                assert got[b, h, i] == nearest_f32(ex), (b, h, i)
    assert got[1, :, nb - 1:].tolist() == [[0.0] * 3] * 2


def test_score_g1_is_plain_matmul_and_linearity_and_scaling():
    rng = np.random.default_rng(5)
    d, nb = 128, 33
    q = rand_bf16(rng, (1, 4, d), 8.0)
    kb = rand_bf16(rng, (1, 4, nb, d), 0.2)
    got = O.score(q, kb, np.array([nb]))                          # G = 1
    ref = np.einsum("hd,hnd->hn", O.bf16_to_f64(q[0]), O.bf16_to_f64(kb[0])) / math.sqrt(d)
    assert np.allclose(got[0], ref, rtol=2e-7, atol=0)
    # G = 4, one KV head: sum over the group == dot with the summed query (exactly, in fp64)
    got4 = O.score(q, kb[:, :1], np.array([nb]))
    qs = O.bf16_to_f64(q[0]).sum(0)
    ref4 = (O.bf16_to_f64(kb[0, 0]) @ qs) * (1.0 / (4 * math.sqrt(d)))
    assert np.array_equal(got4[0, 0], ref4.astype(np.float32))
    # doubling q (exact in bf16: exponent + 1) doubles every score bit-exactly
    q2 = (q + np.uint16(0x0080)).astype(np.uint16)
    assert np.array_equal(O.score(q2, kb[:, :1], np.array([nb])), 2 * got4)


# --------------------------------------------------------------------------------------- top-K
def brute_topk(v, k):
    order = sorted(range(len(v)), key=lambda i: (-float(v[i]), i))
    return sorted(order[:min(k, len(v))])


@pytest.mark.parametrize("n,k", [(1, 1), (7, 3), (16, 16), (16, 40), (100, 13), (257, 64)])
def test_topk_bruteforce_with_ties(n, k):
    rng = np.random.default_rng(n * 31 + k)
    v = rng.integers(-3, 4, n).astype(np.float32) * np.float32(0.25)   # many duplicates
    got = O.topk(v, k)
    assert got.tolist() == brute_topk(v, k)
    sel = set(got.tolist())
    uns = [i for i in range(n) if i not in sel]
    if uns:
        worst = min((float(v[i]), -i) for i in sel)
        best = max((float(v[i]), -i) for i in uns)
        assert worst > best                                          # value desc, index asc


def test_topk_all_equal_neg_zero_and_permutation():
    assert O.topk(np.zeros(10, np.float32), 4).tolist() == [0, 1, 2, 3]
    v = np.array([0.0, -0.0, 0.0, -0.0], np.float32)
    assert O.topk(v, 2).tolist() == [0, 1]                           # -0 == +0: index decides
    rng = np.random.default_rng(7)
    v = rng.standard_normal(50).astype(np.float32)                   # distinct values
    perm = rng.permutation(50)
    a = set(O.topk(v, 9).tolist())
    b = set(perm[O.topk(v[perm], 9)].tolist())
    assert a == b


# ----------------------------------------------------------------------------------------- EMA
def test_ema_constant_step_ramp_closed_forms():
    n, T = 3, 40
    for (alpha, beta, gamma) in [(0.4, 0.3, 0.5), (0.6, 0.6, 0.25), (0.8, 0.1, 0.75)]:
        # constant
        st = O.EmaState(n)
        c = np.array([0.25, -1.0, 3.0], np.float32)
        for _ in range(T):
            O.ema_update(st, c, alpha, beta)
        assert np.array_equal(st.l, c.astype(np.float64)) and not st.v.any()
        assert np.array_equal(O.ema_predict(st, gamma), c)
        # step from (l0, v0 = 0) to constant c
        st = O.EmaState(1)
        l0, cc = 0.5, 2.0
        O.ema_update(st, np.array([l0], np.float32), alpha, beta)     # init l = l0, v = 0
        for t in range(1, T):
            O.ema_update(st, np.array([cc], np.float32), alpha, beta)
            lt = cc + (1 - alpha) ** t * (l0 - cc)
            if alpha != beta:
                vt = beta * (cc - l0) * ((1 - alpha) ** t - (1 - beta) ** t) / (beta - alpha)
            else:
                vt = beta * (cc - l0) * t * (1 - alpha) ** (t - 1)
            assert abs(st.l[0] - lt) < 1e-12 and abs(st.v[0] - vt) < 1e-12, (alpha, beta, t)
        # ramp IS^t = a + s t : lag s(1-alpha)/alpha, v -> s/alpha, prediction error s(1-gamma)/alpha
        st = O.EmaState(1)
        a, s = 1.0, 0.125
        for t in range(400):
            x = np.array([a + s * t], np.float32)
            if t == 399:
                pred = float(O.ema_predict(st, gamma)[0])
            O.ema_update(st, x, alpha, beta)
        assert abs((a + s * 399 - st.l[0]) - s * (1 - alpha) / alpha) < 1e-9
        assert abs(st.v[0] - s / alpha) < 1e-9
        assert abs((a + s * 399 - pred) - s * (1 - gamma) / alpha) < 1e-5


def test_ema_update_uses_old_level_for_trend():
    st = O.EmaState(1)
    O.ema_update(st, np.array([1.0], np.float32), 0.5, 0.5)
    O.ema_update(st, np.array([3.0], np.float32), 0.5, 0.5)
    assert st.l[0] == 2.0 and st.v[0] == 1.0      # v = .5*(3-1) + .5*0 ; with the new l it would be .5
    O.ema_update(st, np.array([3.0], np.float32), 0.5, 0.5)
    assert st.l[0] == 2.5 and st.v[0] == 1.0      # .5*(3-2) + .5*1


def test_ema_reuse_last_topk_special_case_and_scale_invariance():
    """alpha=1, gamma=0, Bud=K  =>  P_t = A_{t-1} (ablation S1)."""
    rng = np.random.default_rng(8)
    n, K = 64, 8
    st, st2 = O.EmaState(n), O.EmaState(n)
    prevA = None
    for t in range(10):
        x = rng.standard_normal(n).astype(np.float32)
        if prevA is not None:
            assert np.array_equal(O.ema_predict_set(st, 0.0, K), prevA)
        O.ema_update(st, x, 1.0, 0.3)
        prevA = O.topk(x, K)
    # new blocks enter without a prediction: state covers only the blocks seen so far
    st = O.EmaState(8)
    O.ema_update(st, np.ones(5, np.float32), 0.4, 0.2)
    assert st.n == 5 and O.ema_predict_set(st, 0.5, 8).tolist() == [0, 1, 2, 3, 4]
    O.ema_update(st, np.arange(7, dtype=np.float32), 0.4, 0.2)
    assert st.n == 7 and st.l[5] == 5.0 and st.v[5] == 0.0 and st.l[6] == 6.0
    # positive power-of-two rescaling of the scores leaves P bit-identical
    st, st2 = O.EmaState(n), O.EmaState(n)
    for t in range(12):
        x = rng.standard_normal(n).astype(np.float32)
        O.ema_update(st, x, 0.6, 0.3)
        O.ema_update(st2, x * np.float32(8.0), 0.6, 0.3)
        assert np.array_equal(O.ema_predict_set(st, 0.75, 12), O.ema_predict_set(st2, 0.75, 12))


# --------------------------------------------------------------------------------- calibration
def test_theta_grid_is_the_papers():
    axes = {}
    for line in open(os.path.join(GOLD, "theta_grid.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, *vals = line.split()
        axes[name] = [float(x) for x in vals]
    grid = O.theta_grid()
    assert len(grid) == int(axes["size"][0]) == 80
    want = [(a, b, g) for a in axes["alpha"] for b in axes["beta"] for g in axes["gamma"]]
    assert grid == want                                   # same doubles as the decimal literals


def _traj(rng, Hkv=2, T=24, N=40, rho=0.9):
    base = rng.standard_normal((Hkv, N)) * 0.5 + 1.0
    rows = []
    x = base.copy()
    for t in range(T):
        x = rho * x + math.sqrt(1 - rho * rho) * (rng.standard_normal((Hkv, N)) * 0.5 + (1 - rho) * 1.0)
        rows.append(np.abs(x) + 0.05)
    return np.stack(rows, axis=1).astype(np.float32)      # [Hkv, T, N], positive


def brute_H(IS, K, Bud, alpha, beta, gamma):
    """Eq. 4 re-typed with python floats, dicts and sorted() — shares nothing with the oracle."""
    Hkv, T, N = IS.shape
    tot, cnt = 0.0, 0
    for h in range(Hkv):
        l, v = {}, {}
        acc = 0.0
        for p in range(T):
            row = [float(x) for x in IS[h, p]]
            if l:
                pred = {i: float(np.float32(l[i] + gamma * v[i])) for i in l}
                P = set(sorted(pred, key=lambda i: (-pred[i], i))[:Bud])
                A = set(sorted(range(N), key=lambda i: (-row[i], i))[:K])
                den = sum(row[i] for i in sorted(A))
                if den > 0:
                    acc += sum(row[i] for i in sorted(A & P)) / den
                    cnt += 1
            for i in range(N):
                if i in l:
                    v[i] = beta * (row[i] - l[i]) + (1 - beta) * v[i]
                    l[i] = alpha * row[i] + (1 - alpha) * l[i]
                else:
                    l[i], v[i] = row[i], 0.0
        tot += acc
    return tot / cnt


def test_calibrate_matches_bruteforce_and_invariants():
    rng = np.random.default_rng(9)
    IS = _traj(rng)
    theta, H, states, H_all = O.calibrate(IS, K=6, budget=8)
    grid = O.theta_grid()
    for ti in (0, 17, 42, 79):
        assert abs(H_all[ti] - brute_H(IS, 6, 8, *grid[ti])) < 1e-12
    assert theta == grid[int(np.argmax(H_all))] and H == H_all.max()
    assert ((H_all >= 0) & (H_all <= 1)).all()
    # gamma = 0 makes beta irrelevant: exact five-way ties
    for a in range(4):
        vals = {H_all[a * 20 + b * 4 + 0] for b in range(5)}
        assert len(vals) == 1
    # the returned state is the state after the last row under theta*
    st = O.EmaState(IS.shape[2])
    for p in range(IS.shape[1]):
        O.ema_update(st, IS[1, p], theta[0], theta[1])
    assert np.array_equal(st.l, states[1].l) and np.array_equal(st.v, states[1].v)
    # budget >= N: everything is predicted, H = 1
    assert O.calibrate(IS, K=6, budget=40)[1] == 1.0


def test_calibrate_constant_trajectory_first_grid_point_and_staircase():
    IS = np.tile(np.linspace(0.1, 1.0, 30, dtype=np.float32), (2, 10, 1))
    theta, H, _, H_all = O.calibrate(IS, K=5, budget=5)
    assert theta == (0.2, 0.1, 0.0) and H == 1.0 and (H_all == 1.0).all()
    # causal staircase: blocks valid at row phi-1 are the only predictable ones
    nv = np.array([10, 10, 20, 20, 30, 30, 30, 30, 30, 30])
    theta, H, states, _ = O.calibrate(IS, K=5, budget=5, n_valid=nv)
    assert states[0].n == 30
    # rows 2 and 4 see new top blocks that had no state yet -> misses -> H < 1
    assert H < 1.0


# ------------------------------------------------------------------------------------ attention
def _dense_ref(q_bits, k_pages, v_pages, table_row, n, bs):
    """Library routine: torch SDPA in fp64 over the gathered dense context."""
    Hq, d = q_bits.shape
    Hkv = k_pages.shape[1]
    nb = (n + bs - 1) // bs
    K = torch.from_numpy(O.bf16_to_f64(k_pages[table_row[:nb]]))       # [nb,Hkv,bs,d]
    V = torch.from_numpy(O.bf16_to_f64(v_pages[table_row[:nb]]))
    K = K.permute(1, 0, 2, 3).reshape(Hkv, nb * bs, d)[:, :n]
    V = V.permute(1, 0, 2, 3).reshape(Hkv, nb * bs, d)[:, :n]
    G = Hq // Hkv
    q = torch.from_numpy(O.bf16_to_f64(q_bits)).reshape(Hkv, G, d)
    out = torch.nn.functional.scaled_dot_product_attention(q[None], K[None], V[None])
    return out[0].reshape(Hq, d).numpy()


def test_attend_all_blocks_is_dense_softmax_attention():
    rng = np.random.default_rng(10)
    k, v, table, lens, bs = _tiny_cache(rng, B=2, Hkv=2, d=16, bs=4, lens=(19, 8))
    q = rand_bf16(rng, (2, 6, 16), 2.0)                               # G = 3
    for b in range(2):
        nb = (lens[b] + bs - 1) // bs
        got = O.attend(q[b], k, v, table[b], lens[b], [range(nb)] * 2, bs)
        assert np.allclose(got, _dense_ref(q[b], k, v, table[b], int(lens[b]), bs), atol=1e-13)


def test_attend_special_cases():
    rng = np.random.default_rng(11)
    k, v, table, lens, bs = _tiny_cache(rng, B=1, Hkv=1, d=8, bs=4, lens=(9,))
    q = rand_bf16(rng, (2, 8), 2.0)
    # one-token context (block 2 holds exactly token 8) -> out = v
    got = O.attend(q, k, v, table[0], 9, [[2]], bs)
    assert np.allclose(got, np.tile(O.bf16_to_f64(v[table[0, 2], 0, 0]), (2, 1)), atol=1e-15)
    # all keys equal -> mean of v
    k2 = k.copy()
    k2[:, :, :, :] = k[0, 0, 0]
    got = O.attend(q, k2, v, table[0], 9, [[0, 1, 2]], bs)
    vv = np.concatenate([O.bf16_to_f64(v[table[0, i], 0, :min(4, 9 - 4 * i)]) for i in range(3)])
    assert np.allclose(got, np.tile(vv.mean(0), (2, 1)), atol=1e-14)
    # empty set -> 0 ; block order irrelevant
    assert not O.attend(q, k, v, table[0], 9, [[]], bs).any()
    a = O.attend(q, k, v, table[0], 9, [[0, 2]], bs)
    b = O.attend(q, k, v, table[0], 9, [[2, 0]], bs)
    assert np.allclose(a, b, atol=1e-15)
    # adding a constant vector to every key shifts all logits of a head equally -> out unchanged
    ki = synth.bits(torch.from_numpy(rng.integers(-4, 5, k.shape).astype(np.float32)).to(torch.bfloat16))
    shift = synth.bits(torch.from_numpy(rng.integers(-3, 4, 8).astype(np.float32)).to(torch.bfloat16))
    ks = synth.bits(torch.from_numpy((O.bf16_to_f64(ki) + O.bf16_to_f64(shift)).astype(np.float32)
                                     ).to(torch.bfloat16))
    a = O.attend(q, ki, v, table[0], 9, [[0, 1, 2]], bs)
    b = O.attend(q, ks, v, table[0], 9, [[0, 1, 2]], bs)
    assert np.allclose(a, b, atol=1e-12)
    # masked tokens (slot >= seq_len) are never read: poison them
    kp, vp = k.copy(), v.copy()
    kp[table[0, 2], :, 1:, :] = 0x7FC0
    vp[table[0, 2], :, 1:, :] = 0x7FC0
    assert np.array_equal(O.attend(q, kp, vp, table[0], 9, [[0, 2]], bs),
                          O.attend(q, k, v, table[0], 9, [[0, 2]], bs))


def test_fold_any_partition_any_order_equals_attend():
    rng = np.random.default_rng(12)
    k, v, table, lens, bs = _tiny_cache(rng, B=1, Hkv=2, d=16, bs=4, lens=(30,))
    q = rand_bf16(rng, (4, 16), 3.0)
    S = [[0, 2, 3, 5, 7], [1, 2, 6]]
    want = O.attend(q, k, v, table[0], 30, S, bs)
    for trial in range(6):
        order = [list(rng.permutation(s)) for s in S]
        cut = [int(rng.integers(0, len(s) + 1)) for s in S]
        first = O.fold(q, k, v, table[0], 30, [o[:c] for o, c in zip(order, cut)], bs)
        both = O.fold(q, k, v, table[0], 30, [o[c:] for o, c in zip(order, cut)], bs, init=first)
        assert np.allclose(O.states_output(both), want, atol=1e-13)
        # l and m are the softmax statistics of the whole set
        for g in range(4):
            h = g // 2
            Kt = np.concatenate([O.block_tokens(k, table[0], 30, h, i, bs) for i in S[h]])
            s = Kt @ O.bf16_to_f64(q[g]) / 4.0
            assert abs(both[g][0] - s.max()) < 1e-14
            assert abs(both[g][1] - np.exp(s - s.max()).sum()) < 1e-12
    # identity element / empty repair
    st = O.fold(q, k, v, table[0], 30, S, bs)
    same = O.fold(q, k, v, table[0], 30, [[], []], bs, init=st)
    assert all(np.array_equal(a[2], b[2]) and a[:2] == b[:2] for a, b in zip(st, same))
    assert O.empty_state(16)[0] == -np.inf and O.empty_state(16)[1] == 0.0


# ------------------------------------------------------------------------------ full PRR step
def _small_layer(policy, seed=13, steps=6):
    cfg = synth.CONFIGS["C0"].scaled(ctx_lo=500, ctx_hi=500, bs=16, K=4, Bud=6, d=32, steps=steps,
                                     T_cal=12, seed=seed)
    inp = synth.make_layer(cfg, 0)
    lay = O.OracleLayer(synth.bits(inp.k_pages), synth.bits(inp.v_pages), inp.block_table.numpy(),
                        inp.seq_lens.numpy(), cfg.bs, cfg.K, cfg.Bud, cfg.Hq, policy)
    return cfg, inp, lay


@pytest.mark.parametrize("policy", [O.DROP, O.RETAIN])
def test_prr_step_speculate_then_repair_equals_definition(policy):
    """Speculative state over P, then Eq. 6-8 over the missed blocks, equals attention over
    A (DROP: only hits are kept from the speculation) / A u P (RETAIN)."""
    cfg, inp, lay = _small_layer(policy)
    lay.calibrate(synth.bits(inp.q_cal))
    hits_seen = miss_seen = 0
    for t in range(cfg.steps):
        lay.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        qb = synth.bits(inp.q_dec[t])
        r = lay.step(qb, update=False)
        for b in range(cfg.B):
            A, P, M, N = r["A"][b], r["P"][b], r["M"][b], r["N"][b]
            for h in range(cfg.Hkv):
                assert set(M[h]) == set(A[h]) - set(P[h]) and set(N[h]) == set(P[h]) - set(A[h])
                assert len(P[h]) == cfg.Bud and len(A[h]) == cfg.K
                hits_seen += len(set(A[h]) & set(P[h])); miss_seen += len(M[h])
            kept = [sorted(set(P[h]) - (set(N[h]) if policy == O.DROP else set())) for h in range(cfg.Hkv)]
            spec = O.fold(qb[b], lay.k, lay.v, lay.table[b], lay.lens[b], kept, cfg.bs)
            rep = O.fold(qb[b], lay.k, lay.v, lay.table[b], lay.lens[b], M, cfg.bs, init=spec)
            assert np.allclose(O.states_output(rep), r["out"][b], atol=1e-13)
            ref_set = A if policy == O.DROP else [np.union1d(a, p) for a, p in zip(A, P)]
            ref = O.attend(qb[b], lay.k, lay.v, lay.table[b], lay.lens[b], ref_set, cfg.bs)
            assert np.array_equal(ref, r["out"][b])
        lay.step(qb)                                           # now with the EMA update
    assert hits_seen > 0 and miss_seen > 0                     # both paths were exercised


def test_prr_step_budget_covers_everything_and_append_keeps_summaries():
    cfg, inp, lay = _small_layer(O.DROP, seed=14, steps=20)
    lay.budget = 10 ** 6
    lay.calibrate(synth.bits(inp.q_cal))
    for t in range(cfg.steps):
        lay.append(synth.bits(inp.k_new[t]), synth.bits(inp.v_new[t]))
        r = lay.step(synth.bits(inp.q_dec[t]))
        nb = lay.n_blocks()[0]
        for h in range(cfg.Hkv):
            # a block that entered this step has no state yet -> can be missed; otherwise M = {}
            assert all(int(i) == nb - 1 for i in r["M"][0][h])
        fresh = O.summarize(lay.k, lay.table, lay.lens, cfg.bs)
        assert np.array_equal(fresh, lay.summ)
    assert lay.lens[0] == 520 and lay.n_blocks()[0] == 33       # crossed a block boundary


def test_synth_is_seeded_and_shaped():
    cfg = synth.CONFIGS["C0"]
    a = synth.make_layer(cfg, 0, steps=4)
    b = synth.make_layer(cfg, 0, steps=4)
    c = synth.make_layer(cfg.scaled(seed=1), 0, steps=4)
    assert torch.equal(a.k_pages.view(torch.int16), b.k_pages.view(torch.int16))
    assert torch.equal(a.q_dec.view(torch.int16), b.q_dec.view(torch.int16))
    assert not torch.equal(a.q_dec.view(torch.int16), c.q_dec.view(torch.int16))
    assert a.k_pages.shape == (66, 2, 64, 64) and a.block_table.shape == (1, 66)
    assert sorted(a.block_table.flatten().tolist()) == list(range(66))
    qn = a.q_dec.float().norm(dim=-1)
    assert torch.allclose(qn, torch.full_like(qn, 8.0), atol=0.05)
    # unwritten slots are poisoned, written ones are finite
    pg = a.block_table[0]
    assert torch.isfinite(a.k_pages[pg[:64].long()].float()).all()
    assert torch.isnan(a.k_pages[pg[64:].long()].float()).all()


# ----------------------------------------------------------------------------------------------
# Quest min / max summaries with the GQA mean query (A.1)
# ----------------------------------------------------------------------------------------------
def _quest_cache(rng, B=2, Hkv=2, d=8, bs=4, lens=(9, 14)):
    nb = max((n + bs - 1) // bs for n in lens)
    n_pages = B * nb
    k = O.f64_to_bf16(rng.standard_normal((n_pages, Hkv, bs, d)))
    table = rng.permutation(n_pages).reshape(B, nb).astype(np.int32)
    return k, table, np.array(lens, dtype=np.int64), bs


def test_quest_summary_is_channelwise_min_max_by_python_loops():
    rng = np.random.default_rng(11)
    k, table, lens, bs = _quest_cache(rng)
    mm = O.summarize_quest(k, table, lens, bs)
    kv = O.bf16_to_f64(k)
    for b in range(2):
        for i in range((lens[b] + bs - 1) // bs):
            n_i = min(bs, lens[b] - i * bs)
            for h in range(2):
                for c in range(8):
                    col = [kv[table[b, i], h, t, c] for t in range(n_i)]
                    assert O.bf16_to_f64(mm[b, h, i, 0, c]) == min(col)
                    assert O.bf16_to_f64(mm[b, h, i, 1, c]) == max(col)


def test_quest_score_by_python_loops_and_mha_form():
    """The formula of A.1 term by term with exact rationals; G = 1 is Quest's own MHA score."""
    from fractions import Fraction
    rng = np.random.default_rng(12)
    k, table, lens, bs = _quest_cache(rng)
    mm = O.summarize_quest(k, table, lens, bs)
    nb = (lens + bs - 1) // bs
    for G in (1, 3):
        q = O.f64_to_bf16(rng.standard_normal((2, 2 * G, 8)))
        got = O.score_quest(q, mm, nb)
        qv, lo, hi = O.bf16_to_f64(q), O.bf16_to_f64(mm[..., 0, :]), O.bf16_to_f64(mm[..., 1, :])
        for b in range(2):
            for h in range(2):
                for p in range(nb[b]):
                    tot = Fraction(0)
                    for i in range(8):
                        qs = sum(Fraction(float(qv[b, h * G + g, i])) for g in range(G))
                        tot += max(qs * Fraction(float(lo[b, h, p, i])), qs * Fraction(float(hi[b, h, p, i])))
                    want = np.float32(float(tot) / (G * np.sqrt(8.0)))
                    assert abs(float(got[b, h, p]) - float(tot) / (G * np.sqrt(8.0))) <= 1e-7 * max(1.0, abs(float(tot)))
                    assert got[b, h, p] == want or abs(float(got[b, h, p]) - float(want)) <= np.spacing(want)


def test_quest_score_reduces_to_mean_score_when_min_equals_max():
    """A block of identical keys (or of one token) has m == M == the mean key: both scores, bit for bit."""
    rng = np.random.default_rng(13)
    k, table, lens, bs = _quest_cache(rng, lens=(8, 13))           # sequence 1: its last block holds one token
    for pg in range(k.shape[0]):
        k[pg, :, :, :] = k[pg, :, :1, :]                           # every block: identical tokens
    q = O.f64_to_bf16(rng.standard_normal((2, 4, 8)))
    nb = (lens + bs - 1) // bs
    s_mean = O.score(q, O.summarize(k, table, lens, bs), nb)
    s_quest = O.score_quest(q, O.summarize_quest(k, table, lens, bs), nb)
    assert np.array_equal(s_mean.view(np.uint32), s_quest.view(np.uint32))


def test_quest_score_is_an_upper_bound_and_scales():
    """Quest's guarantee: s_p >= Qbar . k_t / sqrt d for EVERY token t of the block; doubling q doubles s exactly;
    a wrong sign, a swapped min / max or a dropped channel breaks one of these."""
    rng = np.random.default_rng(14)
    k, table, lens, bs = _quest_cache(rng, d=8, lens=(9, 16))
    mm = O.summarize_quest(k, table, lens, bs)
    nb = (lens + bs - 1) // bs
    G = 2
    q = O.f64_to_bf16(rng.standard_normal((2, 2 * G, 8)))
    s = O.score_quest(q, mm, nb).astype(np.float64)
    qv, kvv = O.bf16_to_f64(q), O.bf16_to_f64(k)
    tight = 0
    for b in range(2):
        for h in range(2):
            qbar = qv[b, h * G:(h + 1) * G].mean(axis=0)
            for p in range(nb[b]):
                n_i = min(bs, lens[b] - p * bs)
                logits = kvv[table[b, p], h, :n_i] @ qbar / np.sqrt(8.0)
                assert s[b, h, p] >= logits.max() - 1e-6
                tight += s[b, h, p] <= logits.max() + 1e-6
    assert tight >= 1                                              # one-token block: the bound is attained
    q2 = O.f64_to_bf16(2.0 * O.bf16_to_f64(q))
    assert np.array_equal((2.0 * O.score_quest(q, mm, nb)).view(np.uint32), O.score_quest(q2, mm, nb).view(np.uint32))
    swapped = mm[:, :, :, ::-1, :]
    assert np.array_equal(O.score_quest(q, swapped, nb).view(np.uint32), O.score_quest(q, mm, nb).view(np.uint32))  # max() is symmetric


def test_oracle_layer_quest_append_keeps_min_max():
    rng = np.random.default_rng(15)
    k, table, lens, bs = _quest_cache(rng, lens=(7, 12))
    table = np.concatenate([table, np.arange(table.size, table.size + 2, dtype=np.int32).reshape(2, 1)], axis=1)
    k = np.concatenate([k, np.zeros((2,) + k.shape[1:], dtype=np.uint16)], axis=0)
    lay = O.OracleLayer(k, k.copy(), table, lens, bs, 2, 2, 4, summary="quest")
    for _ in range(4):
        kn = O.f64_to_bf16(rng.standard_normal((2, 2, 8)))
        lay.append(kn, kn)
    assert np.array_equal(lay.summ, O.summarize_quest(lay.k, lay.table, lay.lens, bs))


# ---- fp8 (e4m3) KV with per-block power-of-two scales (format: DESIGN.md section 10) ----------
def test_e4m3_decode_all_codes_against_torch_and_closed_forms():
    c = np.arange(256, dtype=np.uint8)
    v = O.e4m3_to_f64(c)
    t = torch.from_numpy(c.copy()).view(torch.float8_e4m3fn).to(torch.float32).numpy().astype(np.float64)
    assert np.array_equal(np.isnan(v), np.isnan(t)) and np.isnan(v).sum() == 2          # 0x7f, 0xff only
    assert np.array_equal(v[~np.isnan(v)], t[~np.isnan(t)])
    assert v[0x7E] == 448.0 and v[0xFE] == -448.0 and v[0x01] == 2.0 ** -9 and v[0x08] == 2.0 ** -6
    assert v[0x38] == 1.0 and v[0x3C] == 1.5 and v[0x00] == 0.0 and np.signbit(v[0x80])
    assert np.all(np.diff(v[:127]) > 0)                                                 # what f64_to_e4m3 relies on


def test_e4m3_encode_rne_ties_saturation_round_trip():
    c = np.arange(256, dtype=np.uint8)
    ok = ~np.isnan(O.e4m3_to_f64(c))
    assert np.array_equal(O.f64_to_e4m3(O.e4m3_to_f64(c[ok])), c[ok])                   # every finite code, both zeros
    rng = np.random.default_rng(21)
    x = np.concatenate([rng.standard_normal(20000) * s for s in (0.01, 1.0, 60.0)]).astype(np.float32)
    x = x[np.abs(x) <= 448.0]
    ref = torch.from_numpy(x.copy()).to(torch.float8_e4m3fn).view(torch.uint8).numpy()  # torch rounds to nearest even
    assert np.array_equal(O.f64_to_e4m3(x.astype(np.float64)), ref)
    vals = O.e4m3_to_f64(np.arange(127, dtype=np.uint8))
    mid = (vals[:-1] + vals[1:]) / 2.0                                                  # exact in fp64
    got = O.f64_to_e4m3(mid)
    assert np.all(got % 2 == 0) and np.all((got == np.arange(126)) | (got == np.arange(1, 127)))
    assert np.array_equal(O.f64_to_e4m3(-mid), got | 0x80)
    assert list(O.f64_to_e4m3(np.array([449.0, 1e30, -1e30, np.inf, np.nan, 464.0]))) == [0x7E, 0x7E, 0xFE, 0x7E, 0x7F, 0x7E]
    brute = np.array([np.argmin(np.abs(vals - a)) for a in np.abs(x[:2000]).astype(np.float64)])
    err = np.abs(vals[O.f64_to_e4m3(np.abs(x[:2000]).astype(np.float64))] - np.abs(x[:2000]))
    assert np.all(err <= np.abs(vals[brute] - np.abs(x[:2000])))                        # nearest (brute force over all codes)


def test_pow2_scale_is_the_smallest_that_fits():
    for amax in [448.0, 448.0001, 447.9, 1.0, 0.875, 0.8751, 3.0e-5, 7.0e4, 2.0 ** -20]:
        e = O.pow2_scale_exp(amax)
        assert amax <= 448.0 * 2.0 ** e and amax > 448.0 * 2.0 ** (e - 1)
    assert O.pow2_scale_exp(0.0) == 0


def test_quantize_kv_e4m3_error_bound_and_exact_dequant():
    rng = np.random.default_rng(22)
    bs, Hkv, d = 16, 2, 8
    lens = np.array([37, 64])
    table = rng.permutation(8).astype(np.int32).reshape(2, 4)
    k = O.f64_to_bf16(rng.standard_normal((9, Hkv, bs, d)) * rng.uniform(0.01, 30.0, size=(9, Hkv, 1, 1)))
    k[table[0, 2], :, 5:, :] = 0x7FC0                                                   # NaN in slots past the length
    codes, scale = O.quantize_kv_e4m3(k, table, lens, bs)
    assert codes.dtype == np.uint8 and scale.dtype == np.float32
    assert np.all(codes[8] == 0) and np.all(scale[8] == 1.0)                            # the unmapped page
    assert np.all(codes[table[0, 2], :, 5:, :] == 0)                                    # slots past the length
    assert np.all(codes[table[0, 3]] == 0)                                              # block past the length
    deq = O.bf16_to_f64(O.dequantize_kv_e4m3(codes, scale))
    for b in range(2):
        for i in range(O.n_blocks_of(lens[b], bs)):
            for h in range(Hkv):
                x = O.block_tokens(k, table[b], lens[b], h, i, bs)
                y = deq[table[b, i], h, :x.shape[0]]
                s = float(scale[table[b, i], h])
                assert math.frexp(s)[0] == 0.5                                          # a power of two
                top = np.abs(O.e4m3_to_f64(codes[table[b, i], h, :x.shape[0]])).max()
                assert 224.0 <= top <= 448.0                                            # amax > 224 s rounds to a code >= 224
                assert np.all(np.abs(y - x) <= np.maximum(np.abs(x) * 2.0 ** -4, s * 2.0 ** -10))
    # values that ARE e4m3 codes times the block's scale survive unchanged
    k2 = O.dequantize_kv_e4m3(codes, scale)
    c2, s2 = O.quantize_kv_e4m3(k2, table, np.array([64, 64]), bs)
    live = [table[b, i] for b in range(2) for i in range(O.n_blocks_of(lens[b], bs))]
    assert np.array_equal(O.dequantize_kv_e4m3(c2, s2)[live], k2[live])


def test_oracle_layer_per_sequence_budgets():
    """budget_seq: a sequence's P is the top-budget_seq[b] prediction; None follows the layer's
    budget; a run with budget_seq equal to the layer's budget everywhere is the plain run; a sequence's result does
    not depend on the other sequences' budgets (rows are independent)."""
    rng = np.random.default_rng(31)
    bs, Hkv, d, B = 8, 2, 8, 3
    lens = np.array([61, 80, 47])
    table = rng.permutation(3 * 11).astype(np.int32).reshape(3, 11)
    k = O.f64_to_bf16(rng.standard_normal((34, Hkv, bs, d)))
    v = O.f64_to_bf16(rng.standard_normal((34, Hkv, bs, d)))
    qs = O.f64_to_bf16(rng.standard_normal((5, B, 4, d)))
    def run(budget_seq):
        lay = O.OracleLayer(k, v, table, lens, bs, 3, 5, 4)
        lay.theta = [(0.6, 0.2, 0.5)] * B
        lay.budget_seq = budget_seq
        return [lay.step(qs[t]) for t in range(5)]
    plain, same, mixed = run(None), run([5, 5, None]), run([0, 2, None])
    for t in range(5):
        for b in range(B):
            for h in range(Hkv):
                assert np.array_equal(plain[t]["P"][b][h], same[t]["P"][b][h])
                assert np.array_equal(plain[t]["A"][b][h], mixed[t]["A"][b][h])          # A never depends on the budget
        assert all(len(mixed[t]["P"][0][h]) == 0 for h in range(Hkv))
        assert all(len(mixed[t]["P"][1][h]) <= 2 for h in range(Hkv))
        assert all(np.array_equal(mixed[t]["P"][2][h], plain[t]["P"][2][h]) for h in range(Hkv))
        if t > 0:                                                                       # P_t (budget 2) = the top 2 of P_t (budget 5)
            for h in range(Hkv):
                assert set(mixed[t]["P"][1][h]) <= set(plain[t]["P"][1][h]) and len(mixed[t]["P"][1][h]) == 2
        assert np.array_equal(mixed[t]["out"], plain[t]["out"])                         # DROP: the output is attention over A
