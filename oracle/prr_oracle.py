"""CPU fp64 oracle for the PRR per-layer decode path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this file.  The product (paper_2606_30389_b200/, csrc/, include/) never does,
shares no code, table or constant with it, and has no CPU fallback.

Written from /root/reference/PAPER.md ("Predict, Reuse, and Repair", arxiv 2606.30389); every
function cites the passage it follows.  It is slow and plain on purpose: numpy fp64, library
primitives (matmul, sort) as single steps, no blocking / fusion / reordering beyond what the
definition states.  Inputs are the bf16 bit patterns (uint16) the GPU reads, widened exactly.

What each part is, and what pins it (tests/test_oracle_pins.py; readings Q1..Q15 in DESIGN.md):
  summary        mean-pooled key per block ("compresses each block (e.g., mean)")
                 pins: identical keys -> that key; brute force; power-of-two counts exact
  score          group-aggregated scaled logit against the summary (A.1 PAPER.md:372)
                 pins: exact big-integer dot product; G=1 plain matmul; linearity; x2 scaling bit-exact
  summarize_quest / score_quest   Quest's channel-wise min / max page metadata and its upper-bound score
                 with the GQA mean query, s = sum_i max(Qbar_i m_i, Qbar_i M_i) (A.1)
                 pins: per-channel python loops; G = 1 = Quest's MHA form; m == M -> the mean-summary score
                 bit for bit; s >= the mean query's logit with EVERY token of the block; x2 scaling
  topk           K highest scores, ties -> lower index (BASELINE.json north_star)
                 pins: brute-force python sort incl. duplicates, K>=n, all-equal, permutation invariant
  ema_*          Eq. 2 / Eq. 3, init l=IS, v=0
                 pins: closed forms under constant / step / ramp input; alpha=1,gamma=0 -> P_t = A_{t-1}
  calibrate      Eq. 4 / Eq. 5 over the 80-point grid
                 pins: |grid| = 80; gamma=0 -> beta-independent exact ties; constant trajectory ->
                 first grid point; Bud >= N -> H = 1
  attend         softmax attention over the tokens of a block set
                 pins: all blocks -> dense softmax attention; one token -> v; equal keys -> mean v;
                 key shift invariance; block permutation invariance
  block_state /  per-block (m, l, O) and the Eq. 6-8 fold
  fold           pins: any partition, any order == attend; identity element; M = {} is the identity
  e4m3 codecs /  OCP e4m3 codes, power-of-two per-block scales, quantise / dequantise a paged cache (PAPER.md:319
  quantize_kv    names fp8 as future work; format = DESIGN.md section 10).  pins: all 256 codes and random
                 values against torch.float8_e4m3fn; midpoints tie to even; saturation; round trip; amax of a
                 block lands on a code >= 240/448 of full scale; relative error <= 2^-4; dequantised cache exact in bf16
  prr_step       speculate over P, repair A\\P
                 pins: DROP == attend(A); RETAIN == attend(A u P); Bud = NB -> M = {}
  The paper's published ratios / hit rates (Tables 1-8): PARITY UNPINNED — they depend on models
  and datasets that are not available; nothing in this file is fitted to them.
"""
from __future__ import annotations

import math

import numpy as np

NEG_INF = -np.inf


# ----------------------------------------------------------------------------------------------
# bf16 <-> fp64 (input widening is exact; narrowing is round-to-nearest-even)
# ----------------------------------------------------------------------------------------------
def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    """uint16 bf16 bit patterns -> float64, exactly."""
    b = np.asarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f64_to_bf16(x: np.ndarray) -> np.ndarray:
    """float64 -> bf16 bit patterns, ONE round-to-nearest-even from the fp64 value (finite,
    normal range).  Candidates are the two bf16 neighbours obtained by chopping the fp64
    significand to 7 explicit bits; the nearer wins, a tie goes to the even significand."""
    x = np.asarray(x, dtype=np.float64)
    u = x.view(np.uint64)
    keep = np.uint64(0xFFFFFFFFFFFFFFFF) << np.uint64(52 - 7)
    lo = (u & keep).view(np.float64)                       # toward zero, 8-bit significand
    ulp = np.ldexp(1.0, np.frexp(np.where(lo == 0, 1.0, lo))[1] - 1 - 7)
    ulp = np.where(lo == 0, np.ldexp(1.0, -133), ulp)      # below bf16 normals: smallest step
    hi = lo + np.copysign(ulp, x)                          # away from zero (exact in fp64)
    d_lo = np.abs(x - lo)
    d_hi = np.abs(hi - x)
    with np.errstate(over="ignore"):                       # above the largest bf16 -> inf pattern
        lo_bits = (lo.astype(np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)
        hi_bits = (hi.astype(np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)
    even_lo = (lo_bits & np.uint16(1)) == 0
    take_hi = (d_hi < d_lo) | ((d_hi == d_lo) & ~even_lo)
    return np.where(take_hi, hi_bits, lo_bits).astype(np.uint16)


def f64_to_f32(x: np.ndarray) -> np.ndarray:
    """One RNE to fp32; -0 is canonicalised to +0 (Q4)."""
    y = np.asarray(x, dtype=np.float64).astype(np.float32)
    return np.where(y == 0, np.float32(0.0), y).astype(np.float32)


# ----------------------------------------------------------------------------------------------
# paged KV access
# ----------------------------------------------------------------------------------------------
def n_blocks_of(seq_len: int, bs: int) -> int:
    return (int(seq_len) + bs - 1) // bs


def block_tokens(pages: np.ndarray, table_row: np.ndarray, seq_len: int, h: int, i: int, bs: int):
    """Valid tokens of logical block i of KV head h as float64 [n_i, d]."""
    n_i = min(bs, int(seq_len) - i * bs)
    return bf16_to_f64(pages[int(table_row[i]), h, :n_i, :])


# ----------------------------------------------------------------------------------------------
# 1. summary — PAPER.md:66 "partitions KV tokens into blocks, compresses each block (e.g., mean)"
# ----------------------------------------------------------------------------------------------
def summarize(k_pages, block_table, seq_lens, bs: int, max_blocks: int | None = None) -> np.ndarray:
    """kbar[b,h,i,:] = bf16( mean over the valid tokens of block i ) as uint16 [B,Hkv,max_blocks,d].
    The open (last, partly filled) block is averaged over its valid tokens only (Q2)."""
    B = block_table.shape[0]
    Hkv, d = k_pages.shape[1], k_pages.shape[3]
    mb = block_table.shape[1] if max_blocks is None else max_blocks
    out = np.zeros((B, Hkv, mb, d), dtype=np.uint16)
    for b in range(B):
        for i in range(n_blocks_of(seq_lens[b], bs)):
            for h in range(Hkv):
                k = block_tokens(k_pages, block_table[b], seq_lens[b], h, i, bs)
                out[b, h, i] = f64_to_bf16(k.sum(axis=0) / float(k.shape[0]))
    return out


# ----------------------------------------------------------------------------------------------
# 2. score — PAPER.md:66 "computes compressed attention"; group handled as in A.1:
#    one score per (KV head, block) from the representative query (1/G) sum_g Q_g.
# ----------------------------------------------------------------------------------------------
def score_scale(G: int, d: int) -> float:
    return 1.0 / (G * math.sqrt(float(d)))


def score(q_bits, summ_bits, n_blocks) -> np.ndarray:
    """IS[b,h,i] = fp32( ( sum_{g in group(h)} sum_j q[b,hG+g,j] * kbar[b,h,i,j] ) * c ),
    c = 1/(G sqrt d)  ==  <mean query, mean key> / sqrt(d).  float32 [B,Hkv,max_blocks];
    entries at i >= n_blocks[b] are 0."""
    B, Hq, d = q_bits.shape
    Hkv, mb = summ_bits.shape[1], summ_bits.shape[2]
    G = Hq // Hkv
    c = score_scale(G, d)
    q = bf16_to_f64(q_bits)
    out = np.zeros((B, Hkv, mb), dtype=np.float32)
    for b in range(B):
        nb = int(n_blocks[b])
        for h in range(Hkv):
            kbar = bf16_to_f64(summ_bits[b, h, :nb])            # [nb, d]
            s = np.zeros(nb, dtype=np.float64)
            for g in range(G):
                s = s + kbar @ q[b, h * G + g]
            out[b, h, :nb] = f64_to_f32(s * c)
    return out


# ----------------------------------------------------------------------------------------------
# 2b. Quest scoring extended to GQA — A.1: "we first compute a representative query
#     Qbar = (1/G) sum_g Q_g ... maintain the corresponding channel-wise minimum and maximum key
#     metadata (m_p, M_p) ... the importance score of page p is
#     s_p = sum_i max(Qbar_i m_{p,i}, Qbar_i M_{p,i})".  Scaled like `score` (x 1/sqrt d), so that a
#     block whose min equals its max scores exactly what the mean summary gives.
# ----------------------------------------------------------------------------------------------
def summarize_quest(k_pages, block_table, seq_lens, bs: int, max_blocks: int | None = None) -> np.ndarray:
    """mm[b,h,i,0,:] = channel-wise minimum, mm[b,h,i,1,:] = maximum over the valid tokens of block i, as
    bf16 bit patterns uint16 [B,Hkv,max_blocks,2,d] (min / max of bf16 values are bf16 values: no rounding)."""
    B = block_table.shape[0]
    Hkv, d = k_pages.shape[1], k_pages.shape[3]
    mb = block_table.shape[1] if max_blocks is None else max_blocks
    out = np.zeros((B, Hkv, mb, 2, d), dtype=np.uint16)
    for b in range(B):
        for i in range(n_blocks_of(seq_lens[b], bs)):
            for h in range(Hkv):
                n_i = min(bs, int(seq_lens[b]) - i * bs)
                bits = k_pages[int(block_table[b][i]), h, :n_i, :]          # [n_i, d] uint16
                val = bf16_to_f64(bits)
                out[b, h, i, 0] = bits[np.argmin(val, axis=0), np.arange(d)]
                out[b, h, i, 1] = bits[np.argmax(val, axis=0), np.arange(d)]
    return out


def score_quest(q_bits, mm_bits, n_blocks) -> np.ndarray:
    """s[b,h,p] = fp32( ( sum_i max(qs_i m_{p,i}, qs_i M_{p,i}) ) * c ), qs = sum_{g in group(h)} q_g = G Qbar,
    c = 1/(G sqrt d).  float32 [B,Hkv,max_blocks]; entries at p >= n_blocks[b] are 0."""
    B, Hq, d = q_bits.shape
    Hkv, mb = mm_bits.shape[1], mm_bits.shape[2]
    G = Hq // Hkv
    c = score_scale(G, d)
    q = bf16_to_f64(q_bits)
    out = np.zeros((B, Hkv, mb), dtype=np.float32)
    for b in range(B):
        nb = int(n_blocks[b])
        for h in range(Hkv):
            qs = q[b, h * G:(h + 1) * G].sum(axis=0)                       # [d], exact
            lo = bf16_to_f64(mm_bits[b, h, :nb, 0])                        # [nb, d]
            hi = bf16_to_f64(mm_bits[b, h, :nb, 1])
            s = np.maximum(qs * lo, qs * hi).sum(axis=1)
            out[b, h, :nb] = f64_to_f32(s * c)
    return out


# ----------------------------------------------------------------------------------------------
# 3. top-K — PAPER.md:17 "selecting ... only the top-K ... blocks", A.1 "top-K pages are selected
#    and shared across the group"; ties -> lower block index (BASELINE.json north_star)
# ----------------------------------------------------------------------------------------------
def topk(values: np.ndarray, k: int) -> np.ndarray:
    """Indices of the min(k, n) largest values, order (value desc, index asc); returned ascending."""
    v = np.asarray(values)
    n = v.shape[0]
    order = np.lexsort((np.arange(n), -v.astype(np.float64)))   # last key is primary
    return np.sort(order[:min(k, n)]).astype(np.int32)


# ----------------------------------------------------------------------------------------------
# 4. EMA predictor — PAPER.md:137 (init), Eq. 2 PAPER.md:147 (predict), Eq. 3 PAPER.md:153 (update)
# ----------------------------------------------------------------------------------------------
class EmaState:
    """Level l and trend v per block of one (layer, sequence, KV head); blocks [0, n) have state."""

    def __init__(self, capacity: int):
        self.l = np.zeros(capacity, dtype=np.float64)
        self.v = np.zeros(capacity, dtype=np.float64)
        self.n = 0

    def copy(self) -> "EmaState":
        s = EmaState(self.l.shape[0])
        s.l[:] = self.l
        s.v[:] = self.v
        s.n = self.n
        return s


def ema_predict(st: EmaState, gamma: float) -> np.ndarray:
    """Eq. 2: IS^_i = l_i + gamma * v_i for the blocks that have state; one RNE to fp32."""
    return f64_to_f32(st.l[:st.n] + (gamma * st.v[:st.n]))


def ema_predict_set(st: EmaState, gamma: float, budget: int) -> np.ndarray:
    """P = top-min(Bud, #stateful) blocks by predicted score (Eq. 1 budget)."""
    if st.n == 0:
        return np.zeros(0, dtype=np.int32)
    return topk(ema_predict(st, gamma), budget)


def ema_update(st: EmaState, IS: np.ndarray, alpha: float, beta: float) -> None:
    """Eq. 3 with the score vector of this step (float32 [NB]); both lines use l^{t-1}.
    Blocks seen for the first time are initialised l = IS, v = 0."""
    nb = IS.shape[0]
    x = IS.astype(np.float64)
    n = st.n
    l_old = st.l[:n].copy()
    st.v[:n] = (beta * (x[:n] - l_old)) + ((1.0 - beta) * st.v[:n])
    st.l[:n] = (alpha * x[:n]) + ((1.0 - alpha) * l_old)
    st.l[n:nb] = x[n:nb]
    st.v[n:nb] = 0.0
    st.n = nb


# ----------------------------------------------------------------------------------------------
# 5. calibration — PAPER.md:164-178: Eq. 4 score-weighted hit rate, Eq. 5 argmax over the grid
# ----------------------------------------------------------------------------------------------
def theta_grid():
    """alpha in [0.2,0.8] step 0.2, beta in [0.1,0.5] step 0.1, gamma in [0,0.75] step 0.25
     -> 80 candidates, alpha-major then beta then gamma.  Each value is one
    correctly rounded division so that any implementation holds identical doubles."""
    return [(a / 10.0, b / 10.0, g / 4.0) for a in (2, 4, 6, 8) for b in (1, 2, 3, 4, 5)
            for g in (0, 1, 2, 3)]


def calibrate(IS: np.ndarray, K: int, budget: int, n_valid=None):
    """IS: float32 [Hkv, T, N] prefill trajectory (row phi = score vector at prefill token phi).
    Simulates the predictor for every theta of the grid (Q8): at row phi the stateful blocks are
    those valid at row phi-1; P_phi = predicted top-min(Bud, #stateful); A_phi = top-K of row phi
    over its valid blocks; h_phi = sum_{P n A} IS / sum_A IS, rows with no stateful block or a
    non-positive denominator are skipped; H = mean of h_phi over counted rows and KV heads (Eq. 4).
    Returns (theta*, H*, [EmaState per head after the last row under theta*], H of all 80)."""
    Hkv, T, N = IS.shape
    nv = np.full(T, N, dtype=np.int64) if n_valid is None else np.asarray(n_valid, dtype=np.int64)
    grid = theta_grid()
    A_rows = [[topk(IS[h, p, :nv[p]], K) for p in range(T)] for h in range(Hkv)]
    H_all = np.zeros(len(grid), dtype=np.float64)
    finals = []
    for ti, (alpha, beta, gamma) in enumerate(grid):
        total = 0.0
        count = 0
        states = []
        for h in range(Hkv):
            st = EmaState(N)
            acc = 0.0
            for p in range(T):
                row = IS[h, p, :nv[p]]
                if st.n > 0:
                    P = ema_predict_set(st, gamma, budget)
                    A = A_rows[h][p]
                    den = float(row[A].astype(np.float64).sum())
                    if den > 0.0:
                        hit = np.intersect1d(P, A)
                        num = float(row[hit].astype(np.float64).sum())
                        acc = acc + num / den
                        count += 1
                ema_update(st, row, alpha, beta)
            total = total + acc
            states.append(st)
        H_all[ti] = total / count if count else 0.0
        finals.append(states)
    best = int(np.argmax(H_all))                                  # first maximiser (Eq. 5)
    return grid[best], float(H_all[best]), finals[best], H_all


# ----------------------------------------------------------------------------------------------
# 5b. fp8 (e4m3) KV blocks with per-block scales — PAPER.md:319 names fp8 as future work and fixes no format;
#     DESIGN.md section 10 takes: OCP e4m3 ("fn": no infinities, max 448, NaN = S.1111.111), ONE power-of-two
#     scale per (page, KV head) for K and one for V, the smallest 2^e with amax <= 448 * 2^e, codes =
#     RNE(x / 2^e) saturated to +-448.  A power-of-two scale makes x / 2^e and code * 2^e exact, so the only
#     rounding is the e4m3 one and the dequantised cache is again a bf16 cache: every other function of
#     this file applies to it unchanged.
# ----------------------------------------------------------------------------------------------
def e4m3_to_f64(codes: np.ndarray) -> np.ndarray:
    """uint8 e4m3 codes -> float64, exactly: (-1)^s 2^(E-7) (1 + M/8), E = 0: 2^-6 (M/8); S.1111.111 = NaN."""
    c = np.asarray(codes, dtype=np.uint8).astype(np.int64)
    sgn = np.where(c & 0x80, -1.0, 1.0)
    E = (c >> 3) & 0xF
    M = (c & 0x7).astype(np.float64)
    val = np.where(E == 0, np.ldexp(M / 8.0, -6), np.ldexp(1.0 + M / 8.0, (E - 7).astype(np.int64)))
    val = np.where((E == 15) & ((c & 0x7) == 7), np.nan, val)
    return sgn * val


def f64_to_e4m3(x: np.ndarray) -> np.ndarray:
    """float64 -> e4m3 codes: round to nearest, ties to the even code, |x| beyond 448 saturates to +-448
    (0x7e / 0xfe), NaN -> 0x7f.  The 127 non-negative finite codes are ascending in value, so the nearest
    code is found by searching the table of their values; a tie takes the even code."""
    x = np.asarray(x, dtype=np.float64)
    table = e4m3_to_f64(np.arange(127, dtype=np.uint8))            # 0 .. 448, strictly ascending
    ax = np.minimum(np.abs(np.nan_to_num(x, nan=0.0)), 448.0)
    hi = np.clip(np.searchsorted(table, ax, side="left"), 0, 126)  # first code with value >= ax
    lo = np.maximum(hi - 1, 0)
    d_hi, d_lo = table[hi] - ax, ax - table[lo]
    take_lo = (d_lo < d_hi) | ((d_lo == d_hi) & (lo % 2 == 0))
    code = np.where(take_lo, lo, hi).astype(np.uint8)
    code = np.where(np.signbit(x), code | np.uint8(0x80), code).astype(np.uint8)
    return np.where(np.isnan(x), np.uint8(0x7F), code).astype(np.uint8)


def pow2_scale_exp(amax: float) -> int:
    """Smallest integer e with amax <= 448 * 2^e (0 for an all-zero block)."""
    if not amax > 0.0:
        return 0
    m, x = math.frexp(float(amax))        # amax = m 2^x, 0.5 <= m < 1;  448 = 0.875 * 2^9
    return x - 9 if m <= 0.875 else x - 8


def quantize_kv_e4m3(pages_bits, block_table, seq_lens, bs: int):
    """bf16 pages [n_pages, Hkv, bs, d] -> (codes uint8 of the same shape, scale float32 [n_pages, Hkv]).
    Per (mapped page, KV head): amax over the VALID tokens of the block, scale = 2^e, codes = RNE(x / 2^e).
    Token slots past the sequence length get code 0; pages no sequence maps keep code 0 and scale 1."""
    n_pages, Hkv, _, d = pages_bits.shape
    codes = np.zeros(pages_bits.shape, dtype=np.uint8)
    scale = np.ones((n_pages, Hkv), dtype=np.float32)
    for b in range(block_table.shape[0]):
        for i in range(n_blocks_of(seq_lens[b], bs)):
            pg = int(block_table[b, i])
            for h in range(Hkv):
                x = block_tokens(pages_bits, block_table[b], seq_lens[b], h, i, bs)
                e = pow2_scale_exp(float(np.abs(x).max()))
                scale[pg, h] = np.float32(math.ldexp(1.0, e))
                codes[pg, h, :x.shape[0], :] = f64_to_e4m3(np.ldexp(x, -e))
    return codes, scale


def dequantize_kv_e4m3(codes, scale) -> np.ndarray:
    """codes uint8 [n_pages, Hkv, bs, d], scale float32 [n_pages, Hkv] (powers of two) -> the dequantised
    cache as bf16 bit patterns (exact: 4 significant bits times a power of two)."""
    val = e4m3_to_f64(codes) * scale.astype(np.float64)[:, :, None, None]
    bits = f64_to_bf16(val)
    assert np.array_equal(bf16_to_f64(bits), val), "dequantised fp8 values must be exact in bf16"
    return bits


# ----------------------------------------------------------------------------------------------
# 6. attention over a block set — PAPER.md:66 (sparse attention over the selected blocks), :184
# ----------------------------------------------------------------------------------------------
def attend(q_bits, k_pages, v_pages, table_row, seq_len: int, sets, bs: int) -> np.ndarray:
    """out[g,:] = sum_t softmax_t( q_g . k_t / sqrt d ) v_t over the tokens t < seq_len of the
    blocks in sets[h] (h = KV head of g).  q_bits uint16 [Hq, d] -> float64 [Hq, d].  Empty -> 0."""
    Hq, d = q_bits.shape
    Hkv = k_pages.shape[1]
    G = Hq // Hkv
    q = bf16_to_f64(q_bits)
    out = np.zeros((Hq, d), dtype=np.float64)
    for h in range(Hkv):
        S = [int(i) for i in sets[h]]
        if not S:
            continue
        Kt = np.concatenate([block_tokens(k_pages, table_row, seq_len, h, i, bs) for i in S])
        Vt = np.concatenate([block_tokens(v_pages, table_row, seq_len, h, i, bs) for i in S])
        for g in range(G):
            s = (Kt @ q[h * G + g]) / math.sqrt(float(d))
            p = np.exp(s - s.max())
            out[h * G + g] = (p / p.sum()) @ Vt
    return out


# ----------------------------------------------------------------------------------------------
# 7. partial state and the Eq. 6-8 fold — PAPER.md:184 (speculative kernel also writes l and m),
#    PAPER.md:188-200 (repair recurrence, once per missed block)
# ----------------------------------------------------------------------------------------------
def empty_state(d: int):
    """Identity of the fold: (m, l, O) = (-inf, 0, 0)."""
    return (NEG_INF, 0.0, np.zeros(d, dtype=np.float64))


def fold_block(state, q_vec, Kb, Vb, d: int):
    """One application of Eq. 6-8: fold the tokens of one block (Kb, Vb float64 [n, d]) into the
    running (m, l, O); O is kept normalised, as Eq. 8 writes it."""
    m, l, O = state
    s = (Kb @ q_vec) / math.sqrt(float(d))            # S_{t+1,j}
    m_t = float(s.max())                              # m~
    e = np.exp(s - m_t)
    l_t = float(e.sum())                              # l~
    m_new = max(m, m_t)                               # Eq. 6
    a_old = math.exp(m - m_new) if m != NEG_INF else 0.0
    a_new = math.exp(m_t - m_new)
    l_new = a_old * l + a_new * l_t                   # Eq. 7
    O_new = (a_old * l / l_new) * O + (a_new / l_new) * (e @ Vb)   # Eq. 8
    return (m_new, l_new, O_new)


def fold(q_bits, k_pages, v_pages, table_row, seq_len: int, order, bs: int, init=None):
    """Fold the blocks order[h] (a list per KV head, in that order) into `init` (or the identity)
    for every query head; returns a list of (m, l, O) per query head."""
    Hq, d = q_bits.shape
    Hkv = k_pages.shape[1]
    G = Hq // Hkv
    q = bf16_to_f64(q_bits)
    states = [empty_state(d) for _ in range(Hq)] if init is None else list(init)
    for h in range(Hkv):
        for i in order[h]:
            Kb = block_tokens(k_pages, table_row, seq_len, h, int(i), bs)
            Vb = block_tokens(v_pages, table_row, seq_len, h, int(i), bs)
            for g in range(G):
                states[h * G + g] = fold_block(states[h * G + g], q[h * G + g], Kb, Vb, d)
    return states


def states_output(states) -> np.ndarray:
    return np.stack([O for (_, _, O) in states])


# ----------------------------------------------------------------------------------------------
# 8. one PRR layer-step — PAPER.md:38-42 (predict P, speculate over P while selecting, repair A\P),
#    PAPER.md:102-105 (M = A\P, N = P\A), PAPER.md:121 (the serial fallback = attend over A)
# ----------------------------------------------------------------------------------------------
DROP, RETAIN = 0, 1


def diff_sets(A, P):
    A = np.asarray(A, dtype=np.int32)
    P = np.asarray(P, dtype=np.int32)
    return np.setdiff1d(A, P).astype(np.int32), np.setdiff1d(P, A).astype(np.int32)


class OracleLayer:
    """Plain stateful runner of one layer: paged cache + summaries + EMA state per (seq, KV head).
    Order inside a step (Q10): append, then score/top-K/predict/attend with seq_len including
    the new token, then the EMA update."""

    def __init__(self, k_pages, v_pages, block_table, seq_lens, bs, K, budget, Hq, policy=DROP, summary="mean"):
        self.k = np.array(k_pages, dtype=np.uint16, copy=True)
        self.v = np.array(v_pages, dtype=np.uint16, copy=True)
        self.table = np.asarray(block_table)
        self.lens = np.array(seq_lens, dtype=np.int64, copy=True)
        self.bs, self.K, self.budget, self.Hq, self.policy = bs, K, budget, Hq, policy
        self.B = self.table.shape[0]
        self.Hkv, self.d = self.k.shape[1], self.k.shape[3]
        self.mb = self.table.shape[1]
        self.summary = summary                       # "mean" | "quest" (A.1)
        self.summ = (summarize if summary == "mean" else summarize_quest)(self.k, self.table, self.lens, bs)
        self.ema = [[EmaState(self.mb) for _ in range(self.Hkv)] for _ in range(self.B)]
        self.theta = [(1.0, 1.0, 0.0)] * self.B

    def n_blocks(self):
        return np.array([n_blocks_of(n, self.bs) for n in self.lens], dtype=np.int64)

    def budget_of(self, b: int) -> int:
        """|P| <= delta K (Eq. 1) with delta a per-sequence input: `budget_seq[b]` if set (a list with one
        entry per sequence, None = the layer's budget), else the layer's budget."""
        bs_ = getattr(self, "budget_seq", None)
        return self.budget if bs_ is None or bs_[b] is None else int(bs_[b])

    def scores(self, q_bits):
        return (score if self.summary == "mean" else score_quest)(q_bits, self.summ, self.n_blocks())

    def calibrate(self, q_cal_bits, n_valid=None):
        """Synthetic prefill trajectory (DESIGN.md input recipe): T_cal query rows scored against
        the initial cache; fits theta* per sequence and seeds the EMA state (Q5)."""
        T = q_cal_bits.shape[0]
        nb = self.n_blocks()
        res = []
        for b in range(self.B):
            sfn = score if self.summary == "mean" else score_quest
            IS = np.stack([sfn(q_cal_bits[t, b:b + 1], self.summ[b:b + 1], nb[b:b + 1])[0, :, :nb[b]]
                           for t in range(T)], axis=1)             # [Hkv, T, N]
            theta, H, states, H_all = calibrate(IS, self.K, self.budget, n_valid)
            self.theta[b] = theta
            for h in range(self.Hkv):
                st = EmaState(self.mb)
                st.l[:states[h].n] = states[h].l[:states[h].n]
                st.v[:states[h].n] = states[h].v[:states[h].n]
                st.n = states[h].n
                self.ema[b][h] = st
            res.append((theta, H, H_all, IS))
        return res

    def append(self, k_new_bits, v_new_bits):
        """Write one token per sequence and refresh the open block's summary (a0)."""
        for b in range(self.B):
            pos = int(self.lens[b])
            pg, slot = int(self.table[b, pos // self.bs]), pos % self.bs
            self.k[pg, :, slot, :] = k_new_bits[b]
            self.v[pg, :, slot, :] = v_new_bits[b]
            self.lens[b] = pos + 1
            i = pos // self.bs
            for h in range(self.Hkv):
                if self.summary == "mean":
                    kk = block_tokens(self.k, self.table[b], self.lens[b], h, i, self.bs)
                    self.summ[b, h, i] = f64_to_bf16(kk.sum(axis=0) / float(kk.shape[0]))
                else:
                    kk = block_tokens(self.k, self.table[b], self.lens[b], h, i, self.bs)
                    self.summ[b, h, i, 0] = f64_to_bf16(kk.min(axis=0))          # exact: a min of bf16 values
                    self.summ[b, h, i, 1] = f64_to_bf16(kk.max(axis=0))

    def step(self, q_bits, update=True):
        """q_bits uint16 [B,Hq,d] -> dict(out [B,Hq,d] f64, scores, A, P, M, N per (b,h))."""
        nb = self.n_blocks()
        IS = self.scores(q_bits)
        out = np.zeros((self.B, self.Hq, self.d), dtype=np.float64)
        A_all, P_all, M_all, N_all = [], [], [], []
        for b in range(self.B):
            A_b, P_b, M_b, N_b = [], [], [], []
            _, _, gamma = self.theta[b]
            for h in range(self.Hkv):
                A = topk(IS[b, h, :nb[b]], self.K)
                P = ema_predict_set(self.ema[b][h], gamma, self.budget_of(b))
                M, N = diff_sets(A, P)
                A_b.append(A); P_b.append(P); M_b.append(M); N_b.append(N)
            S = A_b if self.policy == DROP else [np.union1d(a, p) for a, p in zip(A_b, P_b)]
            out[b] = attend(q_bits[b], self.k, self.v, self.table[b], self.lens[b], S, self.bs)
            A_all.append(A_b); P_all.append(P_b); M_all.append(M_b); N_all.append(N_b)
            if update:
                alpha, beta, _ = self.theta[b]
                for h in range(self.Hkv):
                    ema_update(self.ema[b][h], IS[b, h, :nb[b]], alpha, beta)
        return dict(out=out, scores=IS, A=A_all, P=P_all, M=M_all, N=N_all)
