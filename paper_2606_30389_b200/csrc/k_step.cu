// k_step — one PRR layer-step (a1-a8) as ONE persistent launch (Fig. 1, :38-42, :115 Fig. 5).
//
// The paper overlaps speculative attention with selection on two streams; on B200 a layer-step at
// batch 1 moves ~30 MB, i.e. ~5 us of HBM time, so kernel boundaries (2 us each) are the cost that
// matters.  Here the whole step is one grid of #SM CTAs whose WARPS are the workers: each warp owns
// a private shared-memory tile buffer (K and V tile of one block, padded for ldmatrix) and walks
// through the phases below.  Dependencies between warps are device-scope counters (release: data
// stores, __threadfence, atomic; acquire: ld.acquire poll, then L2 (.cg) loads).  Every wait
// targets an EARLIER phase of other warps, all CTAs are co-resident (cooperative launch), so the
// schedule cannot deadlock; waits are bounded anyway and raise ctl[CTL_ERR].
//
//   phase 0  prefetch: cp.async of the warp's first speculative (block, KV head) tile -> all of
//            the step's KV bytes are in flight before anything else happens
//   phase 1  score chunks (a1): 16-byte loads of summary rows, exact fp64 accumulation (Q1)
//   phase 2  row jobs, on the otherwise idle highest-numbered warps:
//              select(row): wait for the row's scores -> exact top-K by range narrowing (a2),
//                           ascending A / bitmask, diff against P (a5) -> M list, publish
//              ema(row):    wait for the row's scores -> Eq. 3 update, Eq. 2 prediction, top-Bud
//                           -> P of the NEXT step into the other parity buffer (a8, a3)
//   phase 3  speculative units (a4): per-block partial state (m, l, O) of every block of P
//   phase 4  repair units (a6): wait for select(row), same partial-state code over M = A\P
//   phase 5  merge items (a7): wait for the row's units, fold hits u M (DROP) or P u M (RETAIN)
//            by Eq. 6-8 with one division at the end
//   exit     last warp resets the counters and flips the layer's P parity
//
// spec = 0 runs the same kernel as the sequential select-then-attend path: P is
// treated as empty, every block of A is a "repair" unit that can only start after selection.
#include <math_constants.h>

#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {

constexpr float LOG2E_F = 1.4426950408889634f;
constexpr uint32_t SPIN_LIMIT = 1u << 22;  // ~0.1-0.5 s of polling, then give up loudly

enum { CTL_EXIT = 0, CTL_ERR = 1, CTL_HDR = 4 };  // then 5 arrays of Rmax words
// ctl arrays: [0] score_done, [1] sel_flag, [2] units_done, [3] units_total, [4] nM

__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// Warp-collective wait until *p >= target.  Lane 0 polls; __syncwarp orders the other lanes.
__device__ __forceinline__ void wait_ge(const uint32_t* p, uint32_t target, uint32_t* err) {
  if ((threadIdx.x & 31) == 0) {
    uint32_t it = 0;
    while (ld_acquire(p) < target) {
      __nanosleep(40);
      if (++it > SPIN_LIMIT) { atomicExch(err, 1u); break; }
    }
  }
  __syncwarp();
}

// Release: every lane has fenced its own stores, then one lane bumps / sets the counter.
__device__ __forceinline__ void signal_add(uint32_t* p, uint32_t v) {
  __threadfence();
  __syncwarp();
  if ((threadIdx.x & 31) == 0) atomicAdd(p, v);
}

__device__ __forceinline__ uint32_t key_at(const float* v, int i) { return score_key(__ldcg(v + i)); }

struct Thr { uint32_t key; int idx; };  // selected(i) <=> key_i > key || (key_i == key && i <= idx)

// ---------------------------------------------------------------------------------------------
// Exact k-th largest of n fp32 values in global memory under the order (value desc, index asc),
// by one warp, as a threshold pair.  Range narrowing on the order-preserving keys: the invariant
// is "the threshold key lies in [lo, lo+span]; `need` of the keys in that range are selected, every
// key above it is".  Each pass counts 16 sub-ranges in packed per-lane counters (no atomics);
// <= 64 survivors are ranked directly; a range of one key value is resolved by index order.
// Integer-only, hence order-independent and bit-exact (Q4).  Requires 1 <= k < n.
// ---------------------------------------------------------------------------------------------
__device__ Thr warp_kth(const float* v, int n, int k, uint32_t* candk, int32_t* candi) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  uint32_t kmin = 0xffffffffu, kmax = 0u;
  for (int i = lane; i < n; i += 32) {
    const uint32_t key = key_at(v, i);
    kmin = min(kmin, key);
    kmax = max(kmax, key);
  }
  uint32_t lo = __reduce_min_sync(FULL, kmin);
  uint32_t span = __reduce_max_sync(FULL, kmax) - lo;
  int need = k, cnt_in = n;
  Thr r;
  for (;;) {
    if (span == 0) {  // all survivors share one key: the `need` lowest indices win
      int base = 0;
      r.key = lo; r.idx = n - 1;
      for (int j0 = 0; j0 < n; j0 += 32) {
        const int i = j0 + lane;
        const uint32_t bal = __ballot_sync(FULL, i < n && key_at(v, i) == lo);
        const int c = __popc(bal);
        if (base + c >= need) { r.idx = j0 + (int)__fns(bal, 0, need - base); break; }
        base += c;
      }
      return r;
    }
    if (cnt_in <= 64) {  // collect the survivors (ascending index) and rank them
      int base = 0;
      for (int j0 = 0; j0 < n; j0 += 32) {
        const int i = j0 + lane;
        const uint32_t key = i < n ? key_at(v, i) : 0u;
        const bool in = i < n && (key - lo) <= span;
        const uint32_t bal = __ballot_sync(FULL, in);
        if (in) {
          const int pos = base + __popc(bal & lt);
          candk[pos] = key;
          candi[pos] = i;
        }
        base += __popc(bal);
      }
      __syncwarp();
      uint32_t wk = 0; int wi = 0; bool won = false;
      for (int e = lane; e < cnt_in; e += 32) {
        const uint32_t ke = candk[e];
        const int ie = candi[e];
        int rank = 0;
        for (int f = 0; f < cnt_in; ++f) {
          const uint32_t kf = candk[f];
          rank += (kf > ke) || (kf == ke && candi[f] < ie);
        }
        if (rank == need - 1) { wk = ke; wi = ie; won = true; }
      }
      const uint32_t bal = __ballot_sync(FULL, won);
      const int src = __ffs(bal) - 1;  // exactly one winner: ranks are a permutation
      r.key = __shfl_sync(FULL, wk, src);
      r.idx = __shfl_sync(FULL, wi, src);
      __syncwarp();
      return r;
    }
    const int sh = max(0, (32 - __clz(span)) - 4);  // (span >> sh) <= 15
    uint32_t cnt[16];
#pragma unroll
    for (int b = 0; b < 16; ++b) cnt[b] = 0;
    for (int i0 = 0; i0 < n; i0 += 32 * 255) {  // 8-bit packed counters: flush every 255 keys per lane
      unsigned long long c0 = 0, c1 = 0;
      const int i1 = min(n, i0 + 32 * 255);
#pragma unroll 4
      for (int i = i0 + lane; i < i1; i += 32) {
        const uint32_t d = key_at(v, i) - lo;
        const uint32_t b = d >> sh;
        const unsigned long long inc = d <= span ? (1ull << ((b & 7u) * 8u)) : 0ull;
        c0 += b < 8u ? inc : 0ull;
        c1 += b < 8u ? 0ull : inc;
      }
#pragma unroll
      for (int b = 0; b < 8; ++b) {
        cnt[b] += (uint32_t)(c0 >> (8 * b)) & 255u;
        cnt[8 + b] += (uint32_t)(c1 >> (8 * b)) & 255u;
      }
    }
#pragma unroll
    for (int b = 0; b < 16; ++b) cnt[b] = __reduce_add_sync(FULL, cnt[b]);
    int acc = 0, bstar = 0, cstar = 0;
    bool found = false;
#pragma unroll
    for (int b = 15; b >= 0; --b) {
      if (!found) {
        if (acc + (int)cnt[b] >= need) { bstar = b; cstar = (int)cnt[b]; found = true; }
        else acc += (int)cnt[b];
      }
    }
    need -= acc;
    cnt_in = cstar;
    const uint32_t off = (uint32_t)bstar << sh;
    const uint32_t width = sh ? ((1u << sh) - 1u) : 0u;
    lo += off;
    span = min(span - off, width);
    if (need == cnt_in) { r.key = lo; r.idx = 0x7fffffff; return r; }  // the whole sub-range is selected
  }
}

__device__ __forceinline__ bool selected(uint32_t key, int i, const Thr& t) {
  return key > t.key || (key == t.key && i <= t.idx);
}

// ---------------------------------------------------------------------------------------------
struct StepArgs {
  const uint16_t* kp; const uint16_t* vp; const int32_t* table; const int32_t* seq_lens;
  const uint16_t* q; const uint4* summ; float* out;
  // layer state (already offset to the layer)
  float* scores; double* ema_l; double* ema_v; int32_t* n_state; const double* theta;
  int32_t* P0; int32_t* P1; int32_t* parity;
  int32_t* setA; int32_t* setM; int32_t* counts;
  // per-step scratch
  uint32_t* maskA; float* pred;
  float* O_spec; float* m_spec; float* l_spec; float* O_rep; float* m_rep; float* l_rep;
  uint32_t* ctl; unsigned long long* stats;
  int B, Hq, Hkv, G, MB, MBw, bs, K, Bud, Rmax, retain, spec, buf_bytes, scr_bytes;
  float scale; double score_c;
};

template <int D, int BS>
struct Tile {
  static constexpr int LD = D + 8;               // padded row stride (elements): ldmatrix conflict-free
  static constexpr int CH = D / 8;               // 16-byte chunks per row
  static constexpr int BYTES = 2 * BS * LD * 2;  // K tile + V tile
  static constexpr int SUB = BS < 64 ? BS : 64;  // tokens per softmax sub-tile
  static constexpr int WFIT = (220 * 1024) / BYTES;
  static constexpr int WMAX = WFIT < 12 ? WFIT : 12;  // warps per CTA (one tile buffer each)
};

// Issue the cp.async loads of one (block, KV head) tile; rows >= valid are zero-filled (unwritten
// cache slots may hold anything, and 0 * NaN must not reach the PV product).  Two commit groups:
// K first, so QK^T can start while V is still in flight.
template <int D, int BS>
__device__ __forceinline__ void tile_load(uint16_t* Ks, const StepArgs& a, int b, int h, int blk, int valid) {
  using T = Tile<D, BS>;
  const int lane = threadIdx.x & 31;
  uint16_t* Vs = Ks + BS * T::LD;
  const size_t page = (size_t)__ldg(a.table + (size_t)b * a.MB + blk);
  const uint16_t* gK = a.kp + ((page * a.Hkv + h) * BS) * (size_t)D;
  const uint16_t* gV = a.vp + ((page * a.Hkv + h) * BS) * (size_t)D;
#pragma unroll 8
  for (int i = 0; i < (BS * T::CH) / 32; ++i) {
    const int c = lane + i * 32, row = c / T::CH, col = c % T::CH;
    uint16_t* dst = Ks + row * T::LD + col * 8;
    if (row < valid) cp_async16(dst, gK + row * D + col * 8);
    else *reinterpret_cast<uint4*>(dst) = make_uint4(0, 0, 0, 0);
  }
  cp_async_commit();
#pragma unroll 8
  for (int i = 0; i < (BS * T::CH) / 32; ++i) {
    const int c = lane + i * 32, row = c / T::CH, col = c % T::CH;
    uint16_t* dst = Vs + row * T::LD + col * 8;
    if (row < valid) cp_async16(dst, gV + row * D + col * 8);
    else *reinterpret_cast<uint4*>(dst) = make_uint4(0, 0, 0, 0);
  }
  cp_async_commit();
}

// Per-block partial state (the forward also writes l and m) by ONE warp from its
// landed tile: S = Q K^T on mma.sync m16n8k16 (the G <= 16 query heads of the group are the M rows,
// zero padded), block-local max / sum with quad shuffles, P V with P as a two-term bf16 split.
// The state is relative to the BLOCK-LOCAL maximum, so a block's partial is the same bits whether
// it was computed speculatively, as a repair, or by the sequential path.
template <int D, int BS>
__device__ __forceinline__ void tile_compute(const uint16_t* Ks, const StepArgs& a, int b, int h, int valid,
                                             float* O, float* Mo, float* Lo, int width, int slot) {
  using T = Tile<D, BS>;
  constexpr int LD = T::LD, SUB = T::SUB, NT8 = SUB / 8;
  const uint16_t* Vs = Ks + BS * LD;
  const int lane = threadIdx.x & 31;
  const int r0 = lane >> 2, tq = lane & 3, mat = lane >> 3, rr = lane & 7;
  const int G = a.G;
  uint32_t qa[D / 16][4];
  {
    const uint16_t* qb = a.q + ((size_t)b * a.Hq + (size_t)h * G) * D;
    const bool v0 = r0 < G, v1 = r0 + 8 < G;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
      const int col = ks * 16 + tq * 2;
      qa[ks][0] = v0 ? __ldg(reinterpret_cast<const uint32_t*>(qb + r0 * D + col)) : 0u;
      qa[ks][1] = v1 ? __ldg(reinterpret_cast<const uint32_t*>(qb + (r0 + 8) * D + col)) : 0u;
      qa[ks][2] = v0 ? __ldg(reinterpret_cast<const uint32_t*>(qb + r0 * D + col + 8)) : 0u;
      qa[ks][3] = v1 ? __ldg(reinterpret_cast<const uint32_t*>(qb + (r0 + 8) * D + col + 8)) : 0u;
    }
  }
  float o[D / 8][4];
#pragma unroll
  for (int dt = 0; dt < D / 8; ++dt)
#pragma unroll
    for (int e = 0; e < 4; ++e) o[dt][e] = 0.f;
  float mrun0 = -CUDART_INF_F, mrun1 = -CUDART_INF_F, l0 = 0.f, l1 = 0.f;  // raw-logit max, denominators
  const float sl2 = a.scale * LOG2E_F;

  cp_async_wait<1>();  // K landed
  __syncwarp();
#pragma unroll
  for (int st = 0; st < BS / SUB; ++st) {
    const int tok0 = st * SUB;
    float s[NT8][4];
#pragma unroll
    for (int nt = 0; nt < NT8; ++nt)
#pragma unroll
      for (int e = 0; e < 4; ++e) s[nt][e] = 0.f;
#pragma unroll
    for (int nt = 0; nt < NT8; ++nt) {
#pragma unroll
      for (int k2 = 0; k2 < D / 32; ++k2) {
        uint32_t b0, b1, b2, b3;
        ldmatrix_x4(b0, b1, b2, b3, Ks + (tok0 + nt * 8 + rr) * LD + k2 * 32 + mat * 8);
        mma_bf16_16816(s[nt], qa[2 * k2], b0, b1);
        mma_bf16_16816(s[nt], qa[2 * k2 + 1], b2, b3);
      }
    }
    float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
#pragma unroll
    for (int nt = 0; nt < NT8; ++nt)
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int tok = tok0 + nt * 8 + tq * 2 + (e & 1);
        if (tok >= valid) s[nt][e] = -CUDART_INF_F;
        if (e < 2) mx0 = fmaxf(mx0, s[nt][e]); else mx1 = fmaxf(mx1, s[nt][e]);
      }
    mx0 = fmaxf(mx0, __shfl_xor_sync(FULL, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(FULL, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(FULL, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(FULL, mx1, 2));
    const float mn0 = fmaxf(mrun0, mx0), mn1 = fmaxf(mrun1, mx1);
    const float off0 = mn0 == -CUDART_INF_F ? 0.f : mn0 * sl2;
    const float off1 = mn1 == -CUDART_INF_F ? 0.f : mn1 * sl2;
    if (BS / SUB > 1 && st > 0) {  // online rescale of what the earlier sub-tile accumulated
      const float f0 = mrun0 == -CUDART_INF_F ? 0.f : ex2(mrun0 * sl2 - off0);
      const float f1 = mrun1 == -CUDART_INF_F ? 0.f : ex2(mrun1 * sl2 - off1);
      l0 *= f0; l1 *= f1;
#pragma unroll
      for (int dt = 0; dt < D / 8; ++dt) { o[dt][0] *= f0; o[dt][1] *= f0; o[dt][2] *= f1; o[dt][3] *= f1; }
    }
    mrun0 = mn0; mrun1 = mn1;
    if (st == 0) { cp_async_wait<0>(); __syncwarp(); }  // V landed
    float ls0 = 0.f, ls1 = 0.f;
#pragma unroll
    for (int kk = 0; kk < SUB / 16; ++kk) {
      uint32_t pa[4], pb[4];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int nt = 2 * kk + u;
        const float p0 = ex2(fmaf(s[nt][0], sl2, -off0)), p1 = ex2(fmaf(s[nt][1], sl2, -off0));
        const float p2 = ex2(fmaf(s[nt][2], sl2, -off1)), p3 = ex2(fmaf(s[nt][3], sl2, -off1));
        const uint32_t h01 = pack_bf16x2(p0, p1), h23 = pack_bf16x2(p2, p3);
        pa[u * 2 + 0] = h01;
        pa[u * 2 + 1] = h23;
        pb[u * 2 + 0] = pack_bf16x2(p0 - bf16_lo(h01), p1 - bf16_hi(h01));
        pb[u * 2 + 1] = pack_bf16x2(p2 - bf16_lo(h23), p3 - bf16_hi(h23));
        ls0 += p0 + p1;
        ls1 += p2 + p3;
      }
#pragma unroll
      for (int d2 = 0; d2 < D / 16; ++d2) {
        uint32_t b0, b1, b2, b3;
        ldmatrix_x4_trans(b0, b1, b2, b3,
                          Vs + (tok0 + kk * 16 + (mat & 1) * 8 + rr) * LD + d2 * 16 + (mat >> 1) * 8);
        mma_bf16_16816(o[2 * d2], pa, b0, b1);
        mma_bf16_16816(o[2 * d2], pb, b0, b1);
        mma_bf16_16816(o[2 * d2 + 1], pa, b2, b3);
        mma_bf16_16816(o[2 * d2 + 1], pb, b2, b3);
      }
    }
    ls0 += __shfl_xor_sync(FULL, ls0, 1);
    ls0 += __shfl_xor_sync(FULL, ls0, 2);
    ls1 += __shfl_xor_sync(FULL, ls1, 1);
    ls1 += __shfl_xor_sync(FULL, ls1, 2);
    l0 += ls0; l1 += ls1;
  }
  __syncwarp();  // every lane is done with the tile: the buffer may be refilled
  const size_t hb = (size_t)b * a.Hq + (size_t)h * G;
  if (r0 < G) {
    const size_t st = (hb + r0) * width + slot;
#pragma unroll
    for (int dt = 0; dt < D / 8; ++dt)
      *reinterpret_cast<float2*>(O + st * D + dt * 8 + tq * 2) = make_float2(o[dt][0], o[dt][1]);
    if (tq == 0) { Mo[st] = mrun0 * a.scale; Lo[st] = l0; }
  }
  if (r0 + 8 < G) {
    const size_t st = (hb + r0 + 8) * width + slot;
#pragma unroll
    for (int dt = 0; dt < D / 8; ++dt)
      *reinterpret_cast<float2*>(O + st * D + dt * 8 + tq * 2) = make_float2(o[dt][2], o[dt][3]);
    if (tq == 0) { Mo[st] = mrun1 * a.scale; Lo[st] = l1; }
  }
}

// ---------------------------------------------------------------------------------------------
// a1: one chunk of summary rows of (b, h): sub-warps of D/8 lanes own a row (one 16-byte load per
// lane), the group's queries are pre-summed per channel in fp64, products and sums are exact (Q1).
template <int D>
__device__ __forceinline__ void score_chunk(const StepArgs& a, int b, int h, int row0, int nb) {
  constexpr int LPR = D / 8, RW = 32 / LPR, UNR = 8;
  const int lane = threadIdx.x & 31, sub = lane / LPR, l = lane % LPR;
  const uint4* rows = a.summ + ((size_t)b * a.Hkv + h) * a.MB * LPR;
  const int rbase = row0 + sub;
  uint4 v[UNR];
#pragma unroll
  for (int u = 0; u < UNR; ++u) {
    const int r = rbase + u * RW;
    v[u] = r < nb ? __ldg(rows + (size_t)r * LPR + l) : make_uint4(0, 0, 0, 0);
  }
  double qs[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) qs[j] = 0.0;
  const uint16_t* qb = a.q + ((size_t)b * a.Hq + (size_t)h * a.G) * D + l * 8;
  for (int g = 0; g < a.G; ++g) {
    const uint4 t = __ldg(reinterpret_cast<const uint4*>(qb + (size_t)g * D));
    const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      qs[2 * j] += (double)bf16_lo(w[j]);
      qs[2 * j + 1] += (double)bf16_hi(w[j]);
    }
  }
  float* out = a.scores + ((size_t)b * a.Hkv + h) * a.MB;
#pragma unroll
  for (int u = 0; u < UNR; ++u) {
    const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
    double acc = 0.0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      acc = fma((double)bf16_lo(w[j]), qs[2 * j], acc);
      acc = fma((double)bf16_hi(w[j]), qs[2 * j + 1], acc);
    }
#pragma unroll
    for (int off = LPR / 2; off >= 1; off >>= 1) acc += __shfl_xor_sync(FULL, acc, off);
    const int r = rbase + u * RW;
    if (l == 0 && r < nb) out[r] = f64_to_score(__dmul_rn(acc, a.score_c));
  }
}

// ---------------------------------------------------------------------------------------------
// a5 preparation, independent of the scores (runs while they are being computed): bitmask of the
// predicted set P in the warp's scratch.  Returns |P|.
__device__ int select_prepare(const StepArgs& a, int row, uint32_t* scr, const int32_t* Pcur) {
  const int lane = threadIdx.x & 31;
  uint32_t* pmask = scr;  // [MBw]
  for (int w = lane; w < a.MBw; w += 32) pmask[w] = 0u;
  __syncwarp();
  int np = 0;
  if (a.spec) {
    const int32_t* P = Pcur + (size_t)row * a.Bud;
    for (int j = lane; j < a.Bud; j += 32) {
      const int blk = __ldg(P + j);
      if (blk >= 0 && blk < a.MB) { atomicOr(&pmask[blk >> 5], 1u << (blk & 31)); ++np; }
    }
  }
  np = __reduce_add_sync(FULL, np);
  __syncwarp();
  return np;
}

// a2 + a5 for one (sequence, KV head) row, by one warp, once the row's scores are complete.
__device__ void job_select(const StepArgs& a, int row, uint32_t* scr, int np) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  const int b = row / a.Hkv;
  const int nb = max(0, min(a.MB, (__ldg(a.seq_lens + b) + a.bs - 1) / a.bs));
  const int nw = (nb + 31) >> 5;
  const uint32_t* pmask = scr;           // [MBw]
  uint32_t* candk = scr + a.MBw;         // [64]
  int32_t* candi = reinterpret_cast<int32_t*>(candk + 64);
  uint32_t* ctl = a.ctl;
  const float* sc = a.scores + (size_t)row * a.MB;
  const int k = min(a.K, nb);
  Thr t;
  t.key = 0u; t.idx = 0x7fffffff;      // k >= n: everything is selected
  if (k < nb) t = warp_kth(sc, nb, k, candk, candi);
  int32_t* A_row = a.setA + (size_t)row * a.K;
  int32_t* M_row = a.setM + (size_t)row * a.K;
  uint32_t* mA = a.maskA + (size_t)row * a.MBw;
  int nA = 0, nM = 0;
  for (int j = 0; j < nw; ++j) {
    const int i = j * 32 + lane;
    const bool sel = i < nb && k > 0 && selected(key_at(sc, i), i, t);
    const uint32_t aw = __ballot_sync(FULL, sel);
    const uint32_t mw = aw & ~pmask[j];
    if (sel) {
      A_row[nA + __popc(aw & lt)] = i;
      if ((mw >> lane) & 1u) M_row[nM + __popc(mw & lt)] = i;
    }
    if (lane == 0) mA[j] = aw;
    nA += __popc(aw);
    nM += __popc(mw);
  }
  for (int j = nA + lane; j < a.K; j += 32) A_row[j] = -1;
  for (int j = nM + lane; j < a.K; j += 32) M_row[j] = -1;
  if (lane == 0) {
    a.counts[row * 3 + 0] = nA;
    a.counts[row * 3 + 1] = np;
    a.counts[row * 3 + 2] = nM;
    if (a.stats) {
      atomicAdd(&a.stats[0], (unsigned long long)nA);
      atomicAdd(&a.stats[1], (unsigned long long)(nA - nM));
      atomicAdd(&a.stats[2], (unsigned long long)nM);
      atomicAdd(&a.stats[3], (unsigned long long)np);
    }
    ctl[CTL_HDR + 3 * a.Rmax + row] = (uint32_t)(np + nM);
    ctl[CTL_HDR + 4 * a.Rmax + row] = (uint32_t)nM;
  }
  signal_add(&ctl[CTL_HDR + 1 * a.Rmax + row], 1u);
}

// a8 + a3 for one row, by one warp: Eq. 3 in non-contracted fp64 (both lines use l^{t-1}; blocks
// scored for the first time get l = IS, v = 0), Eq. 2 rounded once to fp32, then the
// same exact selection for P = top-min(Bud, #stateful) of the next step.
__device__ void job_ema(const StepArgs& a, int row, uint32_t* scr, int32_t* Pnext) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  const int b = row / a.Hkv;
  uint32_t* candk = scr + a.MBw;
  int32_t* candi = reinterpret_cast<int32_t*>(candk + 64);
  double* L = a.ema_l + (size_t)row * a.MB;
  double* V = a.ema_v + (size_t)row * a.MB;
  const double alpha = a.theta[b * 3 + 0], beta = a.theta[b * 3 + 1], gamma = a.theta[b * 3 + 2];
  const double oma = __dsub_rn(1.0, alpha), omb = __dsub_rn(1.0, beta);
  const int n_old = a.n_state[row];
  const int n = max(0, min(a.MB, (__ldg(a.seq_lens + b) + a.bs - 1) / a.bs));
  const int n_new = max(n, n_old);
  const float* sc = a.scores + (size_t)row * a.MB;
  float* pr = a.pred + (size_t)row * a.MB;
  for (int i = lane; i < n_new; i += 32) {
    double ln, vn;
    if (i < n) {
      const double x = (double)__ldcg(sc + i);
      if (i < n_old) {
        const double lo = L[i], vo = V[i];
        vn = __dadd_rn(__dmul_rn(beta, __dsub_rn(x, lo)), __dmul_rn(omb, vo));
        ln = __dadd_rn(__dmul_rn(alpha, x), __dmul_rn(oma, lo));
      } else {
        ln = x;
        vn = 0.0;
      }
      L[i] = ln;
      V[i] = vn;
    } else {
      ln = L[i];
      vn = V[i];
    }
    pr[i] = f64_to_score(__dadd_rn(ln, __dmul_rn(gamma, vn)));
  }
  __syncwarp();
  if (lane == 0) a.n_state[row] = n_new;
  if (a.Bud <= 0) return;
  int32_t* P_row = Pnext + (size_t)row * a.Bud;
  const int k = min(a.Bud, n_new);
  Thr t;
  t.key = 0u; t.idx = 0x7fffffff;
  if (k < n_new) t = warp_kth(pr, n_new, k, candk, candi);
  int cnt = 0;
  for (int j0 = 0; j0 < n_new; j0 += 32) {
    const int i = j0 + lane;
    const bool sel = i < n_new && k > 0 && selected(key_at(pr, i), i, t);
    const uint32_t w = __ballot_sync(FULL, sel);
    if (sel) P_row[cnt + __popc(w & lt)] = i;
    cnt += __popc(w);
  }
  for (int j = cnt + lane; j < a.Bud; j += 32) P_row[j] = -1;
}

// a7 for one (sequence, query head): Eq. 6-8 over the listed partial states, O unnormalised and
// one division at the end.  Entry order is fixed (speculative slots ascending, then repair slots
// ascending), so the result is deterministic; any order is the same real number (Q11).
template <int D>
__device__ void job_merge(const StepArgs& a, int b, int hq, unsigned char* buf, const int32_t* Pcur) {
  constexpr int VEC = D / 32;
  constexpr uint32_t REP = 0x80000000u;
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  const int h = hq / a.G, row = b * a.Hkv + h;
  const size_t hb = (size_t)b * a.Hq + hq;
  const int E = a.Bud + a.K;
  float* ws = reinterpret_cast<float*>(buf);             // [E] m, then weights
  uint32_t* cs = reinterpret_cast<uint32_t*>(buf) + E;   // [E] slot codes (REP bit: repair buffers)
  const int np = a.spec ? __ldcg(a.counts + row * 3 + 1) : 0;
  const int nM = __ldcg(a.counts + row * 3 + 2);
  const uint32_t* mA = a.maskA + (size_t)row * a.MBw;
  const float* Os = a.O_spec + hb * a.Bud * D;
  const float* Or = a.O_rep + hb * a.K * D;
  int n = 0;
  float mx = -CUDART_INF_F;
  // entries: hits (or all of P when retained) ...
  for (int j0 = 0; j0 < np; j0 += 32) {
    const int j = j0 + lane;
    bool use = false;
    if (j < np) {
      const int blk = __ldg(Pcur + (size_t)row * a.Bud + j);
      use = a.retain || ((__ldcg(mA + (blk >> 5)) >> (blk & 31)) & 1u);
    }
    const uint32_t bal = __ballot_sync(FULL, use);
    if (use) {
      const int e = n + __popc(bal & lt);
      const float me = __ldcg(a.m_spec + hb * a.Bud + j);
      ws[e] = me;
      cs[e] = (uint32_t)j;
      mx = fmaxf(mx, me);
    }
    n += __popc(bal);
  }
  // ... then the repaired blocks
  for (int j = lane; j < nM; j += 32) {
    const float me = __ldcg(a.m_rep + hb * a.K + j);
    ws[n + j] = me;
    cs[n + j] = (uint32_t)j | REP;
    mx = fmaxf(mx, me);
  }
  n += nM;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, off));
  __syncwarp();
  float lsum = 0.f;
  for (int e = lane; e < n; e += 32) {
    const float me = ws[e];
    const uint32_t code = cs[e];
    const float w = me == -CUDART_INF_F ? 0.f : ex2((me - mx) * LOG2E_F);
    const float le = (code & REP) ? __ldcg(a.l_rep + hb * a.K + (code & ~REP)) : __ldcg(a.l_spec + hb * a.Bud + code);
    ws[e] = w;
    lsum = fmaf(w, le, lsum);
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) lsum += __shfl_xor_sync(FULL, lsum, off);
  __syncwarp();
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 8
  for (int e = 0; e < n; ++e) {
    const float w = ws[e];
    const uint32_t code = cs[e];
    const float* Op = ((code & REP) ? Or + (size_t)(code & ~REP) * D : Os + (size_t)code * D) + lane * VEC;
    if (VEC == 4) {
      const float4 x = __ldcg(reinterpret_cast<const float4*>(Op));
      acc[0] = fmaf(w, x.x, acc[0]); acc[1] = fmaf(w, x.y, acc[1]);
      acc[2] = fmaf(w, x.z, acc[2]); acc[3] = fmaf(w, x.w, acc[3]);
    } else {
      const float2 x = __ldcg(reinterpret_cast<const float2*>(Op));
      acc[0] = fmaf(w, x.x, acc[0]); acc[1] = fmaf(w, x.y, acc[1]);
    }
  }
  float* o = a.out + hb * D + lane * VEC;
#pragma unroll
  for (int c = 0; c < VEC; ++c) o[c] = lsum > 0.f ? acc[c] / lsum : 0.f;
  __syncwarp();
}

// ---------------------------------------------------------------------------------------------
template <int D, int BS>
__global__ void __launch_bounds__(32 * Tile<D, BS>::WMAX, 1) k_step(const __grid_constant__ StepArgs a) {
  using T = Tile<D, BS>;
  constexpr int LPR = D / 8, CR = (32 / LPR) * 8;  // summary rows per score chunk
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
  const int gw = warp * gridDim.x + blockIdx.x, NW = W * gridDim.x;  // consecutive ids sit on different SMs
  unsigned char* buf = smem_raw + (size_t)warp * (a.buf_bytes + a.scr_bytes);
  uint16_t* Ks = reinterpret_cast<uint16_t*>(buf);
  uint32_t* scr = reinterpret_cast<uint32_t*>(buf + a.buf_bytes);
  uint32_t* ctl = a.ctl;
  uint32_t* score_done = ctl + CTL_HDR;
  uint32_t* sel_flag = ctl + CTL_HDR + a.Rmax;
  uint32_t* units_done = ctl + CTL_HDR + 2 * a.Rmax;
  const uint32_t* units_total = ctl + CTL_HDR + 3 * a.Rmax;
  const uint32_t* nM_g = ctl + CTL_HDR + 4 * a.Rmax;
  const int R = a.B * a.Hkv;
  const int par = *a.parity & 1;
  const int32_t* Pcur = par ? a.P1 : a.P0;
  int32_t* Pnext = par ? a.P0 : a.P1;

  // ---- phase 0: first speculative tile in flight -------------------------------------------
  const int U = a.spec ? R * a.Bud : 0;
  int u = gw;
  int ub = 0, uh = 0, ublk = -1, uvalid = 0;
  auto unit_decode = [&](int unit) {
    const int slot = unit / R, row = unit - slot * R;
    ub = row / a.Hkv; uh = row - ub * a.Hkv;
    ublk = __ldg(Pcur + (size_t)row * a.Bud + slot);
    if (ublk >= a.MB) ublk = -1;
    uvalid = ublk >= 0 ? min(BS, __ldg(a.seq_lens + ub) - ublk * BS) : 0;
  };
  if (u < U) {
    unit_decode(u);
    if (ublk >= 0) tile_load<D, BS>(Ks, a, ub, uh, ublk, uvalid);
  }

  // ---- phase 1: scores ----------------------------------------------------------------------
  {
    const int cpr = (a.MB + CR - 1) / CR;  // chunks per row (static upper bound)
    for (int it = gw; it < R * cpr; it += NW) {
      const int ch = it / R, row = it - ch * R;
      const int b = row / a.Hkv, h = row - b * a.Hkv;
      const int nb = min(a.MB, (__ldg(a.seq_lens + b) + a.bs - 1) / a.bs);
      if (ch * CR >= nb) continue;
      score_chunk<D>(a, b, h, ch * CR, nb);
      signal_add(&score_done[row], 1u);
    }
  }

  // ---- phase 2: row jobs on the highest-numbered warps --------------------------------------
  for (int jj = NW - 1 - gw; jj < 2 * R; jj += NW) {
    const int row = jj < R ? jj : jj - R;
    const int b = row / a.Hkv;
    const int nb = max(0, min(a.MB, (__ldg(a.seq_lens + b) + a.bs - 1) / a.bs));
    int np = 0;
    if (jj < R) np = select_prepare(a, row, scr, Pcur);
    wait_ge(&score_done[row], (uint32_t)((nb + CR - 1) / CR), &ctl[CTL_ERR]);
    if (jj < R) job_select(a, row, scr, np);
    else job_ema(a, row, scr, Pnext);
  }

  // ---- phase 3: speculative units -------------------------------------------------------------
  while (u < U) {
    const int slot = u / R, row = u - slot * R;
    const int cb = ub, chh = uh, cvalid = uvalid;
    const bool real = ublk >= 0;
    if (real) tile_compute<D, BS>(Ks, a, cb, chh, cvalid, a.O_spec, a.m_spec, a.l_spec, a.Bud, slot);
    u += NW;
    if (u < U) {  // refill the buffer before publishing: the next tile's latency starts now
      unit_decode(u);
      if (ublk >= 0) tile_load<D, BS>(Ks, a, ub, uh, ublk, uvalid);
    }
    if (real) signal_add(&units_done[row], 1u);
  }

  // ---- phase 4: repair units --------------------------------------------------------------------
  for (int it = gw; it < R * a.K; it += NW) {
    const int slot = it / R, row = it - slot * R;
    wait_ge(&sel_flag[row], 1u, &ctl[CTL_ERR]);
    const int nM = (int)__ldcg(nM_g + row);
    if (slot >= nM) continue;
    const int b = row / a.Hkv, h = row - b * a.Hkv;
    const int blk = __ldcg(a.setM + (size_t)row * a.K + slot);
    const int valid = min(BS, __ldg(a.seq_lens + b) - blk * BS);
    tile_load<D, BS>(Ks, a, b, h, blk, valid);
    tile_compute<D, BS>(Ks, a, b, h, valid, a.O_rep, a.m_rep, a.l_rep, a.K, slot);
    signal_add(&units_done[row], 1u);
  }

  // ---- phase 5: merge ---------------------------------------------------------------------------
  for (int it = gw; it < a.B * a.Hq; it += NW) {
    const int b = it / a.Hq, hq = it - b * a.Hq;
    const int row = b * a.Hkv + hq / a.G;
    wait_ge(&sel_flag[row], 1u, &ctl[CTL_ERR]);
    wait_ge(&units_done[row], __ldcg(units_total + row), &ctl[CTL_ERR]);
    job_merge<D>(a, b, hq, buf, Pcur);
  }

  // ---- exit: the last warp of the grid resets the step's counters and flips the parity ---------
  __syncwarp();
  uint32_t last = 0;
  if (lane == 0) {
    __threadfence();
    last = atomicAdd(&ctl[CTL_EXIT], 1u) == (uint32_t)(NW - 1);
  }
  last = __shfl_sync(FULL, last, 0);
  if (last) {
    for (int i = lane; i < 5 * a.Rmax; i += 32) ctl[CTL_HDR + i] = 0u;
    if (lane == 0) { ctl[CTL_EXIT] = 0u; *a.parity = par ^ 1; }
  }
}

// ---------------------------------------------------------------------------------------------
template <int D, int BS>
static cudaError_t launch_step_t(prr_ctx* c, const StepArgs& a0, cudaStream_t s) {
  using T = Tile<D, BS>;
  StepArgs a = a0;
  const int merge_bytes = (c->Bud + c->K) * 8;
  a.buf_bytes = (std::max(T::BYTES, merge_bytes) + 15) & ~15;
  a.scr_bytes = ((a.MBw + 128) * 4 + 15) & ~15;
  const int per_warp = a.buf_bytes + a.scr_bytes;
  int W = std::min(T::WMAX, c->smem_optin / per_warp);
  if (W < 1) return cudaErrorInvalidConfiguration;
  const size_t smem = (size_t)W * per_warp;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute((const void*)k_step<D, BS>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(c->n_sm);
  cfg.blockDim = dim3(32 * W);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeCooperative;
  at[0].val.cooperative = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_step<D, BS>, a);
}

int launch_step(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries, float* out,
                int spec, cudaStream_t s) {
  const size_t r = (size_t)kv->layer * c->maxB * c->Hkv;
  StepArgs a{};
  a.kp = (const uint16_t*)kv->k_pages; a.vp = (const uint16_t*)kv->v_pages;
  a.table = kv->block_table; a.seq_lens = kv->seq_lens;
  a.q = (const uint16_t*)q; a.summ = (const uint4*)summaries; a.out = out;
  a.scores = c->scores + r * c->MB;
  a.ema_l = c->ema_l + r * c->MB; a.ema_v = c->ema_v + r * c->MB;
  a.n_state = c->n_state + r;
  a.theta = c->theta + (size_t)kv->layer * c->maxB * 3;
  a.P0 = c->Pbuf[0] + r * c->Bud; a.P1 = c->Pbuf[1] + r * c->Bud; a.parity = c->parity + kv->layer;
  a.setA = c->setA + r * c->K; a.setM = c->setM + r * c->K; a.counts = c->counts + r * 3;
  a.maskA = c->maskA; a.pred = c->pred;
  a.O_spec = c->O_spec; a.m_spec = c->m_spec; a.l_spec = c->l_spec;
  a.O_rep = c->O_rep; a.m_rep = c->m_rep; a.l_rep = c->l_rep;
  a.ctl = c->ctl; a.stats = c->stats;
  a.B = kv->batch; a.Hq = c->Hq; a.Hkv = c->Hkv; a.G = c->G; a.MB = c->MB; a.MBw = (c->MB + 31) / 32;
  a.bs = c->bs; a.K = c->K; a.Bud = c->Bud; a.Rmax = c->maxB * c->Hkv;
  a.retain = c->lay.overpredict_policy == PRR_RETAIN;
  a.spec = (spec && c->Bud > 0) ? 1 : 0;
  a.scale = c->sm_scale; a.score_c = c->score_c;
  cudaError_t e = cudaErrorInvalidValue;
#define PRR_CASE(DD, BB) if (c->D == DD && c->bs == BB) e = launch_step_t<DD, BB>(c, a, s);
  PRR_CASE(128, 64) PRR_CASE(128, 32) PRR_CASE(128, 16) PRR_CASE(128, 128)
  PRR_CASE(64, 64) PRR_CASE(64, 32) PRR_CASE(64, 16) PRR_CASE(64, 128)
#undef PRR_CASE
  c->launches++;
  return e == cudaSuccess ? 0 : (int)e;
}

}  // namespace prr
