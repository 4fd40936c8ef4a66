// k_row — one PRR layer-step (a0-a8) as ONE launch of thread-block CLUSTERS, one cluster per
// (sequence, KV head) row (Fig. 1, :38-42, :115 Fig. 5).
//
// A row -- its summaries, scores, A, P, EMA state, KV blocks and its G query heads -- is independent
// of every other row (selection is per KV head and shared only inside the group), so
// the row is the unit of parallelism and everything BETWEEN the stages of a row stays on chip:
//
//   * the CS CTAs of a cluster split the row's blocks into slices.  Each CTA streams its slice of the
//     summary buffer through its ring of shared-memory buffers (cp.async.bulk), scores it exactly
//     (a1, Q1), applies Eq. 3 / Eq. 2 to its blocks (a8) and sends the order-preserving score keys
//     to EVERY CTA of the cluster and the prediction keys to one (st.async into distributed shared
//     memory, counted by an mbarrier).  No global-memory flag sits between scoring and selection.
//   * every CTA runs the same exact top-K on the gathered keys (a2; redundantly, so nobody has to
//     wait for a broadcast) and therefore knows A, P, hits and M = A\P (a5) without communication.
//   * meanwhile the tile warps compute the CTA's share of the speculative units (a4: predicted
//     blocks dealt round-robin over the CTAs; K and V tiles by TMA in the 128-byte swizzle, one
//     partial state (m, l, O) per block from mma.sync bf16 with the TOKENS as the M dimension).  A
//     partial whose fate is not known yet is parked in a shared-memory slot; once A is known a hit is
//     folded straight into the warp's running state, an over-predicted block is dropped (PRR_DROP)
//     and predicted blocks whose tile has not been requested yet are not requested at all.
//   * missed blocks are repaired (a6) by the CTA that owns their slice: same tile code.
//   * merge (a7): each CTA folds its hit slots and its warps' running states per query head (Eq. 6-8),
//     sends the result to the head's reducer CTA (st.async again), which normalises and writes out.
//   * one CTA of the cluster ranks the prediction keys: P of the next step (a3), off the critical path.
//
// spec = 0 runs the same kernel as the sequential select-then-attend path: P is
// treated as empty and every block of A is a "repair" unit that can only start after selection.
#include <cuda.h>
#include <math_constants.h>

#include <algorithm>
#include <cstring>

#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {
namespace cluster {  // (k_step.cu has its own tile / selection code: keep the two apart)

constexpr float LOG2E_F = 1.4426950408889634f;
constexpr int NWARP = 12, NTHR = 32 * NWARP;
constexpr int SCW = 8;             // warps 0 .. 7 score, then rank the true top-K together
constexpr int GA0 = 0, GAW = 4;    // group A, warps 0 .. 3, then: the true top-K, the diff, Eq. 3 / Eq. 2, the lists, the next
                                   //   prediction, the merge
constexpr int TW0 = 4, NTW = 7;    // tile warps 4 .. 10: 8 .. 10 from the start, 4 .. 7 once they have scored and selected
constexpr int LDW = 11;            // loader warp: predicted-set staging, then every bulk / TMA request
constexpr int NBMAX = 12;          // ring buffers at most
constexpr int HB = 256;            // histogram buckets of a selection pass (shared memory is better spent on slots)
constexpr int CAND = 128;          // survivors that are ranked directly
constexpr unsigned long long WAIT_NS = 200000000ull;  // every wait gives up loudly after 0.2 s

enum { CTL_EXIT = 0, CTL_ERR = 1, CTL_EPOCH = 2, CTL_SITE = 4 };

struct RowArgs {
  alignas(64) CUtensorMap mapK;  // bf16 [rows = n_pages*Hkv*bs, d], box [ST, 64], 128-byte swizzle
  alignas(64) CUtensorMap mapV;
  const int32_t* table; const int32_t* seq_lens;
  // fused append (a0): app = 1 -> seq_lens holds the lengths BEFORE the append, every length below is +1
  const uint16_t* k_new; const uint16_t* v_new; uint16_t* kp_w; uint16_t* vp_w; uint4* summ_w; double* open_sum;
  int32_t* seq_lens_w; int app;
  const uint16_t* q; const uint4* summ; float* out;
  // layer state (already offset to the layer)
  float* scores; double* ema_l; double* ema_v; int32_t* n_state; const double* theta;
  int32_t* P0; int32_t* P1; int32_t* parity;
  int32_t* setA; int32_t* setM; int32_t* counts;
  uint32_t* ctl; unsigned long long* stats; unsigned long long* tl;
  int B, Hq, Hkv, G, MB, MBw, bs, K, Bud, retain, spec, cut;
  int recompute;  // ablation S1: any miss in the row -> the speculative result is discarded, all of A is fetched
  int BudMax;  // the largest run-time budget among the launch's sequences (sizes the parking slots)
  int CS, NBUF, NSLOT, UCAP, HL, SLMAX, NBH, BudSel;  // BudSel <= Bud: the run-time budget of the NEXT prediction
  // dynamic shared memory offsets (bytes)
  int o_keys, o_pkeys, o_hist, o_plist, o_pmask, o_amask, o_offs, o_tslice, o_sc, o_units, o_cand, o_red,
      o_slots, o_slotblk, o_recv, o_end;
  float scale; double score_c;
  uint32_t* done_host; uint32_t done_seq;  // host-visible completion word (mapped host memory) and its value, or null
  const int32_t* bud_seq;  // per sequence of the layer: 0 = the layer's budget, v > 0 = budget v - 1 (prr_set_budget_seq)
};

// ---------------------------------------------------------------------------------------------
// cluster / distributed-shared-memory primitives
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory"); }
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
// store into another CTA's shared memory; the bytes are counted by that CTA's mbarrier (complete_tx)
__device__ __forceinline__ void st_async_v4(uint32_t raddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t rbar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1,%2,%3,%4}, [%5];\n"
               ::"r"(raddr), "r"(a), "r"(b), "r"(c), "r"(d), "r"(rbar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cl(unsigned long long* bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }\n"
      : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return done != 0;
}
__device__ __forceinline__ bool mbar_test_wait(unsigned long long* bar, uint32_t parity) {  // (does not suspend)
  uint32_t done;
  asm volatile(
      "{ .reg .pred p; mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }\n"
      : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return done != 0;
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;\n" : "=r"(d) : "r"(a));
  return d;
}
__device__ __forceinline__ unsigned long long gtime() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;\n" : "=l"(t));
  return t;
}
// Bounded waits: a dependency that never arrives raises ctl[CTL_ERR] (prr_check) instead of hanging; the
// first site that gave up is kept in ctl[CTL_SITE] (site code | CTA << 8 | warp << 20).
__device__ __noinline__ void wait_fail(uint32_t* err, uint32_t site) {
  atomicCAS(err + (CTL_SITE - CTL_ERR), 0u, site | (blockIdx.x << 8) | ((threadIdx.x >> 5) << 20));
  atomicExch(err, 1u);
}
__device__ __forceinline__ void wait_bar(unsigned long long* bar, uint32_t parity, uint32_t* err, uint32_t site) {
  if (mbar_try_wait_cl(bar, parity)) return;
  const unsigned long long t0 = gtime();
  uint32_t it = 0;
  while (!mbar_try_wait_cl(bar, parity))
    if ((++it & 1023u) == 0 && (long long)(gtime() - t0) > (long long)WAIT_NS) { wait_fail(err, site); return; }
}
__device__ __forceinline__ void wait_flag(const volatile int* f, uint32_t* err, uint32_t site) {
  if (*f) return;
  const unsigned long long t0 = gtime();
  uint32_t it = 0;
  while (!*f) {
    __nanosleep(32);
    if ((++it & 1023u) == 0 && (long long)(gtime() - t0) > (long long)WAIT_NS) { wait_fail(err, site); return; }
  }
}

// ---------------------------------------------------------------------------------------------
// Exact selection by a GROUP of warps (a named barrier): the k-th largest of n keys under the order
// (key desc, index asc) as a threshold pair; integer-only, hence order-independent and bit-exact (Q4).
// ---------------------------------------------------------------------------------------------
struct Thr { uint32_t key; int idx; };  // selected(i) <=> key_i > key || (key_i == key && i <= idx)
__device__ __forceinline__ bool selected(uint32_t key, int i, const Thr& t) {
  return key > t.key || (key == t.key && i <= t.idx);
}
struct Grp {
  int tid, nt, wid, nw, bar;
  __device__ __forceinline__ void sync() const { asm volatile("bar.sync %0, %1;\n" ::"r"(bar), "r"(nt) : "memory"); }
};
struct SelMem {
  uint32_t* hist;            // [HB], zero on entry to and exit from grp_kth
  uint32_t* red;             // [nw * 2 + 16]: per-warp slots, then 16 decision words
  unsigned long long* cand;  // [CAND]
  uint32_t* offs;            // [MBw] emission offsets
};

// Highest bucket b with  sum_{b' >= b} hist[b'] >= need  (1 <= need <= total); `above` = the count
// in the buckets over b.  Thread t owns the buckets [HB-(t+1)per, HB-t*per): a prefix scan over
// threads is a suffix scan over buckets.  Every thread zeroes what it read and returns the triple.
__device__ __noinline__ void grp_pick(const Grp& g, const SelMem& m, int need, int& bstar, int& cstar, int& above) {
  const int lane = threadIdx.x & 31;
  uint32_t* dec = m.red + g.nw * 2;
  const int per = (HB + g.nt - 1) / g.nt;
  const int hi = max(0, HB - g.tid * per), lo = max(0, hi - per);
  uint32_t sum = 0;
#pragma unroll 4
  for (int b = lo; b < hi; ++b) sum += m.hist[b];
  uint32_t incl = sum;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const uint32_t x = __shfl_up_sync(FULL, incl, off);
    if (lane >= off) incl += x;
  }
  if (lane == 31) m.red[g.wid] = incl;
  g.sync();
#pragma unroll 1
  for (int w = 0; w < g.wid; ++w) incl += m.red[w];
  const uint32_t excl = incl - sum;
  if ((int)excl < need && need <= (int)incl) {  // the crossing is in this thread's buckets (exactly one thread)
    uint32_t acc = excl;
#pragma unroll 1
    for (int b = hi - 1; b >= lo; --b) {
      const uint32_t c = m.hist[b];
      if ((int)(acc + c) >= need) { dec[0] = (uint32_t)b; dec[1] = c; dec[2] = acc; break; }
      acc += c;
    }
  }
#pragma unroll 1
  for (int b = lo; b < hi; ++b) m.hist[b] = 0u;
  g.sync();
  bstar = (int)dec[0]; cstar = (int)dec[1]; above = (int)dec[2];
  g.sync();  // dec and red are reused by the caller
}

// keys[0 .. n), 1 <= k < n.
__device__ __noinline__ Thr grp_kth_cont(const uint32_t* keys, int n, const Grp& g, const SelMem& m, uint32_t lo, uint32_t span,
                                         int need, int cnt_in, unsigned long long* tl);
__device__ __noinline__ Thr grp_kth(const uint32_t* keys, int n, int k, const Grp& g, const SelMem& m, unsigned long long* tl = nullptr) {
  const int lane = threadIdx.x & 31;
  // the exact key range of the row
  uint32_t kmin = 0xffffffffu, kmax = 0u;
#pragma unroll 4
  for (int i = g.tid; i < n; i += g.nt) { const uint32_t x = keys[i]; kmin = min(kmin, x); kmax = max(kmax, x); }
  kmin = __reduce_min_sync(FULL, kmin);
  kmax = __reduce_max_sync(FULL, kmax);
  if (lane == 0) { m.red[g.wid * 2] = kmin; m.red[g.wid * 2 + 1] = kmax; }
  g.sync();
#pragma unroll 1
  for (int w = 0; w < g.nw; ++w) { kmin = min(kmin, m.red[w * 2]); kmax = max(kmax, m.red[w * 2 + 1]); }
  g.sync();
  if (tl && lane == 0) tl[10] = gtime();
  return grp_kth_cont(keys, n, g, m, kmin, kmax - kmin, k, n, tl);
}
// Range narrowing from a known state (see the invariant below).
__device__ __noinline__ Thr grp_kth_cont(const uint32_t* keys, int n, const Grp& g, const SelMem& m, uint32_t lo, uint32_t span,
                                         int need, int cnt_in, unsigned long long* tl) {
  const int lane = threadIdx.x & 31;
  uint32_t* dec = m.red + g.nw * 2;
  Thr r;
  // invariant: the threshold key lies in [lo, lo+span]; `need` of the cnt_in keys in that range are
  // selected, every key above it is
  for (;;) {
    if (span == 0) {  // all survivors share one key: the `need` lowest indices win
      if (g.wid == 0) {
        int base = 0, idx = n - 1;
#pragma unroll 1
        for (int j0 = 0; j0 < n; j0 += 32) {
          const int i = j0 + lane;
          const uint32_t bal = __ballot_sync(FULL, i < n && keys[i] == lo);
          const int c = __popc(bal);
          if (base + c >= need) { idx = j0 + (int)__fns(bal, 0, need - base); break; }
          base += c;
        }
        if (lane == 0) { dec[5] = lo; dec[6] = (uint32_t)idx; }
      }
      g.sync();
      r.key = dec[5]; r.idx = (int)dec[6];
      g.sync();
      return r;
    }
    if (cnt_in <= CAND) {  // collect the survivors (any order) and rank them: word = key << 32 | ~index
      if (g.tid == 0) dec[7] = 0u;
      g.sync();
#pragma unroll 4
      for (int i = g.tid; i < n; i += g.nt) {
        const uint32_t key = keys[i];
        if ((key - lo) <= span) {
          const uint32_t pos = atomicAdd(&dec[7], 1u);
          m.cand[pos] = ((unsigned long long)key << 32) | (uint32_t)~i;
        }
      }
      g.sync();
      if (tl && lane == 0) tl[13] = gtime();
#pragma unroll 1
      for (int e = g.tid; e < cnt_in; e += g.nt) {
        const unsigned long long ce = m.cand[e];
        uint32_t rank = 0;
#pragma unroll 4
        for (int f = 0; f < cnt_in; ++f) rank += m.cand[f] > ce;
        if ((int)rank == need - 1) { dec[5] = (uint32_t)(ce >> 32); dec[6] = ~(uint32_t)ce; }  // exactly one
      }
      g.sync();
      r.key = dec[5]; r.idx = (int)dec[6];
      g.sync();
      return r;
    }
    const int sh = max(0, (32 - __clz(span)) - 8);  // (span >> sh) < HB
#pragma unroll 4
    for (int i = g.tid; i < n; i += g.nt) {
      const uint32_t d = keys[i] - lo;
      if (d <= span) atomicAdd(&m.hist[d >> sh], 1u);
    }
    g.sync();
    if (tl && lane == 0 && tl[11] == 0) tl[11] = gtime();
    int bstar, cstar, above;
    grp_pick(g, m, need, bstar, cstar, above);
    if (tl && lane == 0 && tl[12] == 0) tl[12] = gtime();
    need -= above;
    cnt_in = cstar;
    const uint32_t off = (uint32_t)bstar << sh;
    const uint32_t width = sh ? ((1u << sh) - 1u) : 0u;
    lo += off;
    span = min(span - off, width);
    if (need == cnt_in) { r.key = lo; r.idx = 0x7fffffff; return r; }  // the whole sub-range is selected
  }
}

// Bitmask of the selected blocks into mask[0 .. nwd) (shared), one ballot per 32 blocks.
__device__ __noinline__ void grp_mask(const uint32_t* keys, int n, int k, const Thr& t, const Grp& g, uint32_t* mask) {
  const int lane = threadIdx.x & 31;
  const int nwd = (n + 31) >> 5;
#pragma unroll 2
  for (int w = g.wid; w < nwd; w += g.nw) {
    const int i = w * 32 + lane;
    const bool sel = i < n && k > 0 && selected(keys[i], i, t);
    const uint32_t bal = __ballot_sync(FULL, sel);
    if (lane == 0) mask[w] = bal;
  }
}

__device__ __forceinline__ float key_value(uint32_t key) {  // inverse of score_key (key 0 = NaN -> -inf)
  if (key == 0u) return -CUDART_INF_F;
  return __uint_as_float((key & 0x80000000u) ? (key & 0x7fffffffu) : ~key);
}

// Selection without a histogram, for k <= NT (a group of NT threads, n <= NT * KR keys in registers).
// Shared-memory atomics run at about one lane per clock, so a histogram over all n keys costs n clocks;
// plain compares on registers do not.  A LOWER BOUND of the k-th largest key comes from the per-thread
// maxima: if every warp's r-th largest thread maximum is >= L, with r = ceil(k / #warps), then at least k
// distinct keys are >= L.  Only the keys >= L (a few more than k) are collected (one atomic per warp)
// and ranked exactly.  Everything is branch-free predicated code: a lone warp issues a dependent
// instruction every ~10 clocks, so the instruction count per thread IS the latency.
constexpr int CANDX = 512;
// The k-th largest (1-based) of the c <= CANDX survivors in m.cand (key << 32 | ~index), all with keys in
// [klo, khi]: 256 buckets linear in VALUE over that range (order-preserving keys are logarithmic in value),
// one atomic per survivor, suffix pick, then the handful of survivors in the crossing bucket are ranked.
template <int NT>
__device__ __forceinline__ void cand_kth(int c, int k, uint32_t klo, uint32_t khi, const Grp& g, const SelMem& m,
                                         uint32_t& tkey, int& tidx) {
  constexpr int NW = NT / 32, NBK = 256, PER = NBK / NT, CPT = CANDX / NT;
  static_assert(PER >= 1 && CPT >= 1, "group of at most 256 threads");
  const int lane = threadIdx.x & 31;
  uint32_t* dec = m.red + NW * 2;
  unsigned long long* cand2 = m.cand + CANDX;  // [64]
  const float vlo = key_value(klo), vhi = key_value(khi);
  const float inv = (float)NBK / (vhi - vlo);
  const bool lin = (vhi > vlo) & (inv < CUDART_INF_F) & (vlo > -CUDART_INF_F);  // (uniform) else: one bucket
  unsigned long long ce[CPT];
  int bk[CPT];
#pragma unroll
  for (int q = 0; q < CPT; ++q) {
    const int j = g.tid + q * NT;
    ce[q] = m.cand[min(j, c - 1)];
    bk[q] = lin ? min(NBK - 1, max(0, (int)((key_value((uint32_t)(ce[q] >> 32)) - vlo) * inv))) : 0;
    if (j < c) atomicAdd(&m.hist[bk[q]], 1u);
  }
  if (g.tid == 0) dec[7] = 0u;
  g.sync();
  // suffix pick: thread t owns the buckets [NBK - (t+1) PER, NBK - t PER)
  const int hb = NBK - g.tid * PER;
  uint32_t hv[PER], sum = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { hv[q] = m.hist[hb - 1 - q]; sum += hv[q]; }
  uint32_t incl = sum;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const uint32_t x = __shfl_up_sync(FULL, incl, off);
    incl += lane >= off ? x : 0u;
  }
  if (lane == 31) m.red[g.wid] = incl;
  g.sync();
#pragma unroll
  for (int w = 0; w < NW; ++w) incl += w < g.wid ? m.red[w] : 0u;
  uint32_t acc = incl - sum;
#pragma unroll
  for (int q = 0; q < PER; ++q) {
    if (((int)acc < k) & (k <= (int)(acc + hv[q]))) { dec[0] = (uint32_t)(hb - 1 - q); dec[1] = hv[q]; dec[2] = acc; }  // exactly one
    acc += hv[q];
    m.hist[hb - 1 - q] = 0u;
  }
  g.sync();
  const int bstar = (int)dec[0], cstar = (int)dec[1], need = k - (int)dec[2];
#pragma unroll
  for (int q = 0; q < CPT; ++q)
    if ((g.tid + q * NT < c) & (bk[q] == bstar)) {
      const uint32_t pos = atomicAdd(&dec[7], 1u);
      if (pos < 64u) cand2[pos] = ce[q];
    }
  g.sync();
  if (cstar <= 64) {
    if (g.tid < cstar) {
      const unsigned long long x = cand2[g.tid];
      int rk = 0;
#pragma unroll 4
      for (int f = 0; f < cstar; ++f) rk += cand2[f] > x;
      if (rk == need - 1) { dec[5] = (uint32_t)(x >> 32); dec[6] = ~(uint32_t)x; }  // exactly one
    }
  } else {  // (heavy ties inside one bucket) every survivor against all
#pragma unroll 1
    for (int j = g.tid; j < c; j += NT) {
      const unsigned long long x = m.cand[j];
      int rk = 0;
#pragma unroll 4
      for (int f = 0; f < c; ++f) rk += m.cand[f] > x;
      if (rk == k - 1) { dec[5] = (uint32_t)(x >> 32); dec[6] = ~(uint32_t)x; }
    }
  }
  g.sync();
  tkey = dec[5]; tidx = (int)dec[6];
}
__device__ __forceinline__ bool selected_bf(uint32_t key, int i, uint32_t tkey, int tidx) {  // (no short circuit)
  return (key > tkey) | ((key == tkey) & (i <= tidx));
}
#ifndef PRR_SEL_INLINE
#define PRR_SEL_INLINE __forceinline__
#endif
template <int NT, int KR>
__device__ PRR_SEL_INLINE void grp_select_v3(const uint32_t* keys, int n, int k, const Grp& g, const SelMem& m, uint32_t* mask,
                                           unsigned long long* tl) {
  constexpr int NW = NT / 32;
  const int lane = threadIdx.x & 31;
  uint32_t* dec = m.red + NW * 2;
  uint32_t kr[KR];
  uint32_t tmax = 0u;
#pragma unroll
  for (int e = 0; e < KR; ++e) {
    const int i = g.tid + e * NT;
    kr[e] = keys[min(i, n - 1)];
    kr[e] = i < n ? kr[e] : 0u;
    tmax = max(tmax, kr[e]);
  }
  uint32_t tkey = 0u;
  int tidx = 0x7fffffff;  // k >= n: everything is selected
  if (k < n) {            // (uniform)
    // the warp's r-th largest thread maximum: r rounds of (max, retire its lowest lane)
    const int r = (k + NW - 1) / NW;  // <= 32
    uint32_t v = tmax, wl = 0u;
#pragma unroll 1
    for (int j = 0; j < r; ++j) {
      wl = __reduce_max_sync(FULL, v);
      const uint32_t eq = __ballot_sync(FULL, v == wl);
      v = lane == __ffs(eq) - 1 ? 0u : v;
    }
    const uint32_t wmax = __reduce_max_sync(FULL, tmax);
    if (lane == 0) { m.red[g.wid] = wl; m.red[NW + g.wid] = wmax; }
    if (g.tid == 0) dec[7] = 0u;
    g.sync();
    uint32_t L = 0xffffffffu, KMAX = 0u;
#pragma unroll
    for (int w = 0; w < NW; ++w) { L = min(L, m.red[w]); KMAX = max(KMAX, m.red[NW + w]); }
    if (tl && lane == 0) tl[10] = gtime();
    // survivors: per-thread bitmask, warp prefix, ONE atomic per warp
    unsigned long long cm = 0ull;
#pragma unroll
    for (int e = 0; e < KR; ++e) cm |= (unsigned long long)((g.tid + e * NT < n) & (kr[e] >= L)) << e;
    const int mine = __popcll(cm);
    int incl = mine;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int x = __shfl_up_sync(FULL, incl, off);
      incl += lane >= off ? x : 0;
    }
    int base = 0;
    if (lane == 31) base = (int)atomicAdd(&dec[7], (uint32_t)incl);
    base = __shfl_sync(FULL, base, 31) + incl - mine;
#pragma unroll
    for (int e = 0; e < KR; ++e)
      if ((cm >> e) & 1ull) {
        if (base < CANDX) m.cand[base] = ((unsigned long long)kr[e] << 32) | (uint32_t)~(g.tid + e * NT);
        ++base;
      }
    g.sync();
    const int c = (int)dec[7];
    if (tl && lane == 0) tl[11] = gtime();
    if (c > CANDX) {  // (ties, or rows shorter than the group): the generic narrowing
      g.sync();
      const Thr t = grp_kth(keys, n, k, g, m, nullptr);
      tkey = t.key; tidx = t.idx;
    } else {
      g.sync();  // (red / dec are reused)
      cand_kth<NT>(c, k, L, KMAX, g, m, tkey, tidx);
    }
  }
  if (tl && lane == 0) tl[14] = gtime();
  const int nwd = (n + 31) >> 5;
  const bool kpos = k > 0;
#pragma unroll
  for (int e = 0; e < KR; ++e) {  // lanes of a warp hold 32 consecutive blocks: one mask word per (warp, e)
    const int i = g.tid + e * NT, w = e * NW + g.wid;
    const uint32_t bal = __ballot_sync(FULL, (i < n) & kpos & selected_bf(kr[e], i, tkey, tidx));
    if ((lane == 0) & (w < nwd)) mask[w] = bal;
  }
}

// Ordered emission from a bitmask: the set bits ascending into list[width] (padded with -1); with
// Mlist != null also the set bits NOT in pmask (ascending, padded to widthM).  Returns (nA << 16) | nM.
__device__ __noinline__ uint32_t grp_emit(const uint32_t* mask, const uint32_t* pmask, int n, const Grp& g, const SelMem& m,
                             int32_t* list, int width, int32_t* Mlist, int widthM) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  const int nwd = (n + 31) >> 5;
  uint32_t* dec = m.red + g.nw * 2;
  if (g.wid == 0) {
    uint32_t carry = 0;
#pragma unroll 1
    for (int w0 = 0; w0 < nwd; w0 += 32) {
      const int w = w0 + lane;
      const uint32_t aw = w < nwd ? mask[w] : 0u;
      const uint32_t mw = (Mlist && w < nwd) ? (aw & ~pmask[w]) : 0u;
      const uint32_t v = ((uint32_t)__popc(aw) << 16) | (uint32_t)__popc(mw);
      uint32_t incl = v;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const uint32_t x = __shfl_up_sync(FULL, incl, off);
        if (lane >= off) incl += x;
      }
      if (w < nwd) m.offs[w] = carry + incl - v;
      carry += __shfl_sync(FULL, incl, 31);
    }
    if (lane == 0) dec[3] = carry;
  }
  g.sync();
#pragma unroll 2
  for (int w = g.wid; w < nwd; w += g.nw) {
    const uint32_t aw = mask[w];
    const uint32_t off = m.offs[w];
    const int i = w * 32 + lane;
    if ((aw >> lane) & 1u) {
      list[(off >> 16) + __popc(aw & lt)] = i;
      if (Mlist) {
        const uint32_t mw = aw & ~pmask[w];
        if ((mw >> lane) & 1u) Mlist[(off & 0xffffu) + __popc(mw & lt)] = i;
      }
    }
  }
  const uint32_t tot = dec[3];
#pragma unroll 1
  for (int j = (int)(tot >> 16) + g.tid; j < width; j += g.nt) list[j] = -1;
  if (Mlist)
#pragma unroll 1
    for (int j = (int)(tot & 0xffffu) + g.tid; j < widthM; j += g.nt) Mlist[j] = -1;
  g.sync();
  return tot;
}

// ---------------------------------------------------------------------------------------------
// Tiles.  Shared-memory image of one (block, KV head, sub-tile) as the copy engine writes it: the
// K half then the V half, each D/64 boxes of [ST rows x 128 bytes] in the 128-byte swizzle (the
// 16-byte chunk c of row r sits at chunk c ^ (r & 7)), so ldmatrix is conflict-free without padding.
// ---------------------------------------------------------------------------------------------
template <int D, int ST>
struct Tile {
  static constexpr int NBOX = D / 64;
  static constexpr int BOX_BYTES = ST * 128;
  static constexpr int HALF = NBOX * BOX_BYTES;  // = ST * D * 2
  static constexpr int BYTES = 2 * HALF;         // K tile + V tile
  static constexpr int CHR = BYTES / (D * 2);    // summary rows one buffer holds (= 2 ST)
  __device__ static __forceinline__ const unsigned char* at(const unsigned char* half, int r, int c) {
    return half + (c >> 3) * BOX_BYTES + r * 128 + (((c & 7) ^ (r & 7)) << 4);
  }
};

// Partial state of one landed tile for the (<= 8) query heads of one pass (the forward
// also writes l and m), by ONE warp: S^T = K Q^T on mma.sync m16n8k16 with the TOKENS as the M rows
// (a 16-token slab of the tile is the A operand straight from the swizzled image, the query heads
// are the 8 columns of B, zero padded), tile-local max / sum over the token dimension with
// shuffles, then O^T = V^T P^T with V^T through ldmatrix.trans and P^T from the score fragments by
// movmatrix (P as a two-term bf16 split).  Per thread: heads g = 2 (lane % 4) + {0, 1};
// o[dt] = O^T[d = 16 dt + lane / 4 (+ 8)][g].  m in log2 units of the scaled logit.
template <int D, int ST>
__device__ __forceinline__ void tile_partial(const unsigned char* Ks, unsigned long long* barK, unsigned long long* barV,
                                             uint32_t par, const uint32_t (&qb)[D / 16][2], int valid, float sl2,
                                             const uint16_t* patch_k, const uint16_t* patch_v, bool first_pass,
                                             float (&o)[D / 16][4], float (&mt)[2], float (&lt)[2], uint32_t* err,
                                             unsigned long long* tl = nullptr) {
  using T = Tile<D, ST>;
  constexpr int NM = ST / 16;
  const unsigned char* Vs = Ks + T::HALF;
  const int lane = threadIdx.x & 31;
  const int r0 = lane >> 2;
  float s[NM][4];
#pragma unroll
  for (int m = 0; m < NM; ++m)
#pragma unroll
    for (int e = 0; e < 4; ++e) s[m][e] = 0.f;
#pragma unroll
  for (int dt = 0; dt < D / 16; ++dt)
#pragma unroll
    for (int e = 0; e < 4; ++e) o[dt][e] = 0.f;

  if (first_pass) {
    wait_bar(barK, par, err, 1);  // K landed
    if (patch_k) {  // fused append: the token appended by this launch is not in the cache yet
      if (lane < D / 8)
        *reinterpret_cast<uint4*>(const_cast<unsigned char*>(T::at(Ks, valid - 1, lane))) =
            __ldg(reinterpret_cast<const uint4*>(patch_k) + lane);
      __syncwarp();
    }
  }
  {
    const int arow = (lane & 7) + ((lane >> 3) & 1) * 8, acol = lane >> 4;
#pragma unroll
    for (int m = 0; m < NM; ++m)
#pragma unroll
      for (int k16 = 0; k16 < D / 16; ++k16) {
        uint32_t a[4];
        ldmatrix_x4(a[0], a[1], a[2], a[3], T::at(Ks, m * 16 + arow, k16 * 2 + acol));
        mma_bf16_16816(s[m], a, qb[k16][0], qb[k16][1]);
      }
  }
  float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
#pragma unroll
  for (int m = 0; m < NM; ++m) {
    const int t0 = m * 16 + r0;
    if (t0 >= valid) { s[m][0] = -CUDART_INF_F; s[m][1] = -CUDART_INF_F; }
    if (t0 + 8 >= valid) { s[m][2] = -CUDART_INF_F; s[m][3] = -CUDART_INF_F; }
    mx0 = fmaxf(mx0, fmaxf(s[m][0], s[m][2]));
    mx1 = fmaxf(mx1, fmaxf(s[m][1], s[m][3]));
  }
#pragma unroll
  for (int off = 4; off <= 16; off <<= 1) {
    mx0 = fmaxf(mx0, __shfl_xor_sync(FULL, mx0, off));
    mx1 = fmaxf(mx1, __shfl_xor_sync(FULL, mx1, off));
  }
  const unsigned long long tq1 = tl ? gtime() : 0ull;
  const float off0 = mx0 * sl2, off1 = mx1 * sl2;  // valid >= 1: the maxima are finite
  mt[0] = off0; mt[1] = off1;
  if (first_pass) {
    wait_bar(barV, par, err, 2);  // V landed
    if (patch_v) {
      if (lane < D / 8)
        *reinterpret_cast<uint4*>(const_cast<unsigned char*>(T::at(Vs, valid - 1, lane))) =
            __ldg(reinterpret_cast<const uint4*>(patch_v) + lane);
    }
    if (valid < ST) {  // open block: 0 * (whatever an unwritten slot holds) must not reach P V
      for (int i = lane; i < (ST - valid) * T::NBOX * 8; i += 32) {
        const int r = valid + i / (T::NBOX * 8), c = i % (T::NBOX * 8);
        *reinterpret_cast<uint4*>(const_cast<unsigned char*>(Vs) + (c >> 3) * T::BOX_BYTES + r * 128 + ((c & 7) << 4)) =
            make_uint4(0, 0, 0, 0);
      }
    }
    __syncwarp();
  }
  float ls0 = 0.f, ls1 = 0.f;
  const int vrow = (lane & 7) + ((lane >> 4) & 1) * 8, vcol = (lane >> 3) & 1;
#pragma unroll
  for (int kk = 0; kk < NM; ++kk) {
    const float p0 = ex2(fmaf(s[kk][0], sl2, -off0)), p1 = ex2(fmaf(s[kk][1], sl2, -off1));
    const float p2 = ex2(fmaf(s[kk][2], sl2, -off0)), p3 = ex2(fmaf(s[kk][3], sl2, -off1));
    ls0 += p0 + p2;
    ls1 += p1 + p3;
    const uint32_t h01 = pack_bf16x2(p0, p1), h23 = pack_bf16x2(p2, p3);
    const uint32_t l01 = pack_bf16x2(p0 - bf16_lo(h01), p1 - bf16_hi(h01));
    const uint32_t l23 = pack_bf16x2(p2 - bf16_lo(h23), p3 - bf16_hi(h23));
    const uint32_t bh0 = movmatrix_trans(h01), bh1 = movmatrix_trans(h23);
    const uint32_t bl0 = movmatrix_trans(l01), bl1 = movmatrix_trans(l23);
#pragma unroll
    for (int dt = 0; dt < D / 16; ++dt) {
      uint32_t a[4];
      ldmatrix_x4_trans(a[0], a[1], a[2], a[3], T::at(Vs, kk * 16 + vrow, dt * 2 + vcol));
      mma_bf16_16816(o[dt], a, bh0, bh1);
      mma_bf16_16816(o[dt], a, bl0, bl1);
    }
  }
#pragma unroll
  for (int off = 4; off <= 16; off <<= 1) {
    ls0 += __shfl_xor_sync(FULL, ls0, off);
    ls1 += __shfl_xor_sync(FULL, ls1, off);
  }
  lt[0] = ls0; lt[1] = ls1;
  if (tl && (threadIdx.x & 31) == 0) { const unsigned long long tq2 = gtime(); tl[2] += tq2 - tq1; tl[1] = tq1; }
}

// State image in shared memory (slots, warp running states, received partials): per query head
// [m, l, -, -, O[D]] = D + 4 floats; the stride keeps the fragment stores conflict-free.
// Fold a tile partial into a state (Eq. 6-8, unnormalised) or overwrite the state with it.
template <int D>
__device__ __forceinline__ void state_put(float* st, int G, int pass, const float (&o)[D / 16][4], const float (&mt)[2],
                                          const float (&lt)[2], bool fold) {
  const int lane = threadIdx.x & 31, r0 = lane >> 2, tq = lane & 3;
  float al[2] = {0.f, 0.f}, be[2] = {1.f, 1.f}, mn[2], ln[2];
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const int g = pass * 8 + tq * 2 + j;
    mn[j] = mt[j]; ln[j] = lt[j];
    if (fold && g < G) {
      const float mo = st[g * (D + 4)], lo = st[g * (D + 4) + 1];
      mn[j] = fmaxf(mo, mt[j]);
      al[j] = mo == -CUDART_INF_F ? 0.f : ex2(mo - mn[j]);
      be[j] = ex2(mt[j] - mn[j]);
      ln[j] = al[j] * lo + be[j] * lt[j];
    }
  }
  __syncwarp();  // every lane has read the old m, l
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const int g = pass * 8 + tq * 2 + j;
    if (g < G) {
      float* row = st + g * (D + 4) + 4;
#pragma unroll
      for (int dt = 0; dt < D / 16; ++dt) {
        const int d0 = dt * 16 + r0;
        if (fold) {
          row[d0] = al[j] * row[d0] + be[j] * o[dt][j];
          row[d0 + 8] = al[j] * row[d0 + 8] + be[j] * o[dt][2 + j];
        } else {
          row[d0] = o[dt][j];
          row[d0 + 8] = o[dt][2 + j];
        }
      }
      if (r0 == 0) { st[g * (D + 4)] = mn[j]; st[g * (D + 4) + 1] = ln[j]; }
    }
  }
  __syncwarp();
}

struct Sh {  // static shared memory
  unsigned long long fullK[NBMAX], fullV[NBMAX], empty[NBMAX];
  unsigned long long bar_keys, bar_pred, bar_red, bar_tw;
  volatile int q_issued, q_total, q_final, sel_done, spec_ready, n_rep;
  int t_next, n_slots, rep_cnt, ring_pos;
  int chunk_cnt[NBMAX];
  volatile int pos_unit[NBMAX];
  volatile int patch_ready;  // the open block's new summary row is in patch_row
  volatile int no_hits;      // S1: the row had a miss, nothing speculative is used
  int miss_cnt;
  alignas(16) uint32_t patch_row[64];
};

// ---------------------------------------------------------------------------------------------
template <int D, int ST>
__global__ void __launch_bounds__(NTHR, 1) k_row(const __grid_constant__ RowArgs a) {
  using T = Tile<D, ST>;
  constexpr int LPR = D / 8, RW = 32 / LPR;  // lanes per summary row, rows per warp trip
  constexpr int CHR = T::CHR;                // summary rows per ring buffer
  constexpr int RPW = CHR / SCW;             // rows of a chunk per scoring warp (4, 8 or 16)
  constexpr int NV = RPW / RW;               // rows per lane group and chunk
  constexpr int SW = D + 4;                  // state row stride (floats)
  static_assert(RPW * SCW == CHR && RPW % 4 == 0 && NV >= 1 && NV <= LPR, "chunk rows must fit the scoring warps");
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ Sh sh;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int CS = a.CS, NBUF = a.NBUF;
  const uint32_t rank = CS > 1 ? cluster_ctarank() : 0u;
  uint32_t* err = a.ctl + CTL_ERR;

  unsigned char* ring = smem;
  uint32_t* keys = reinterpret_cast<uint32_t*>(smem + a.o_keys);
  uint32_t* pkeys = reinterpret_cast<uint32_t*>(smem + a.o_pkeys);
  uint32_t* hist = reinterpret_cast<uint32_t*>(smem + a.o_hist);  // [2][HB]
  int32_t* plist = reinterpret_cast<int32_t*>(smem + a.o_plist);
  uint32_t* pmask = reinterpret_cast<uint32_t*>(smem + a.o_pmask);
  uint32_t* amask = reinterpret_cast<uint32_t*>(smem + a.o_amask);
  uint32_t* offs = reinterpret_cast<uint32_t*>(smem + a.o_offs);  // [2][MBw]
  int32_t* tslice = reinterpret_cast<int32_t*>(smem + a.o_tslice);
  float* scs = reinterpret_cast<float*>(smem + a.o_sc);
  int2* units = reinterpret_cast<int2*>(smem + a.o_units);
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(smem + a.o_cand);  // [2][CAND]
  uint32_t* red = reinterpret_cast<uint32_t*>(smem + a.o_red);                        // [2][32]
  float* slots = reinterpret_cast<float*>(smem + a.o_slots);  // [NSLOT + NTW][G][SW]
  int32_t* slotblk = reinterpret_cast<int32_t*>(smem + a.o_slotblk);
  float* recv = reinterpret_cast<float*>(smem + a.o_recv);    // [CS][HL][SW]
  const int SLOTF = a.G * SW;  // floats per state image

  if (tid == 0) {
    for (int i = 0; i < NBUF; ++i) { mbar_init(&sh.fullK[i], 1); mbar_init(&sh.fullV[i], 1); mbar_init(&sh.empty[i], 1); }
    mbar_init(&sh.bar_keys, 1); mbar_init(&sh.bar_pred, 1); mbar_init(&sh.bar_red, 1); mbar_init(&sh.bar_tw, NTW);
    mbar_fence_init();
    sh.ring_pos = 0;
    for (int i = 0; i < NBMAX; ++i) sh.chunk_cnt[i] = 0;
    sh.q_issued = 0;
  }
  for (int i = tid; i < 2 * HB; i += NTHR) hist[i] = 0u;
  // per-row state; set again at the end of a row if another one follows (nothing here depends on the row,
  // so the first requests of a row wait for nothing but its length)
  auto row_init = [&]() {
    if (tid == 0) {
      sh.q_total = 0; sh.q_final = 0; sh.sel_done = 0; sh.spec_ready = 0; sh.n_rep = 0;
      sh.t_next = 0; sh.n_slots = 0; sh.rep_cnt = 0; sh.patch_ready = 0; sh.no_hits = 0; sh.miss_cnt = 0;
    }
    for (int i = tid; i < NTW * SLOTF; i += NTHR) slots[(size_t)a.NSLOT * SLOTF + i] = (i % SW) == 0 ? -CUDART_INF_F : 0.f;
    for (int i = tid; i < a.MBw; i += NTHR) { pmask[i] = 0u; amask[i] = 0u; }
  };
  row_init();
  __syncthreads();
  if (CS > 1) cluster_arrive();
  // Programmatic dependent launch: let the next step's grid be scheduled (its CTAs take the SMs as
  // ours exit and its launch latency hides behind this step); wait for the previous step's grid to
  // have completed before the first global access.  No-ops without the launch attribute.
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  {  // While the previous grid drains: prefetch (L2 is the point of coherence, so a line the previous grid
     // still writes is simply written again) the first row's summary slice, EMA state, table slice and
     // the control words.  Every one of these is otherwise a TLB miss + HBM miss at the head of the step.
    const int row = blockIdx.x / CS;
    if (row < a.B * a.Hkv) {
      const int b = row / a.Hkv;
      const int nb4 = (a.NBH + 3) & ~3;
      const int slice = ((nb4 + CS - 1) / CS + 3) & ~3;
      const int s0 = min(nb4, (int)rank * slice), s1 = min(min(nb4, s0 + slice), a.MB);
      const size_t rowoff = (size_t)row * a.MB;
      auto pf = [](const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); };
      const char* sp = reinterpret_cast<const char*>(a.summ) + (rowoff + s0) * (size_t)(D * 2);
      const int nline = max(0, s1 - s0) * (D * 2) / 128;
#pragma unroll 1
      for (int i = tid; i < nline; i += NTHR) pf(sp + (size_t)i * 128);
      const int nl8 = (max(0, s1 - s0) * 8 + 127) / 128;  // lines of a double-per-block slice
      if (warp == 8)
#pragma unroll 1
        for (int i = lane; i < nl8; i += 32) { pf(reinterpret_cast<const char*>(a.ema_l + rowoff + s0) + i * 128); pf(reinterpret_cast<const char*>(a.ema_v + rowoff + s0) + i * 128); }
      if (warp == 9)
#pragma unroll 1
        for (int i = lane; i < (nl8 + 1) / 2; i += 32) pf(reinterpret_cast<const char*>(a.table + (size_t)b * a.MB + s0) + i * 128);
      if (warp == 10) {
#pragma unroll 1
        for (int i = lane; i < (a.Bud * 4 + 127) / 128; i += 32) { pf(reinterpret_cast<const char*>(a.P0 + (size_t)row * a.Bud) + i * 128); pf(reinterpret_cast<const char*>(a.P1 + (size_t)row * a.Bud) + i * 128); }
        if (lane == 0) { pf(a.seq_lens + b); pf(a.parity); pf(a.theta + b * 3); pf(a.n_state + row); pf(a.ctl); }
        if (a.app && lane >= 8 && lane < 8 + (D * 8 + 127) / 128) pf(reinterpret_cast<const char*>(a.open_sum + (size_t)row * D) + (lane - 8) * 128);
        if (a.app && lane >= 20 && lane < 20 + (D * 2 + 127) / 128) {
          pf(reinterpret_cast<const char*>(a.k_new + (size_t)row * D) + (lane - 20) * 128);
          pf(reinterpret_cast<const char*>(a.v_new + (size_t)row * D) + (lane - 20) * 128);
        }
      }
    }
  }
  asm volatile("griddepcontrol.wait;\n" ::: "memory");
  // phase stamps are collected in shared memory and written out at exit (the buffer is host memory);
  // the progress mark [15] goes out at once, so it survives a hang
  __shared__ unsigned long long stamps[NWARP][16];
  unsigned long long* tlg = a.tl ? a.tl + ((size_t)blockIdx.x * NWARP + warp) * 16 : nullptr;
  unsigned long long* tl = a.tl ? stamps[warp] : nullptr;
#define MARK(code) do { if (tlg && lane == 0) tlg[15] = (unsigned long long)(code); } while (0)
  if (tl && lane == 0) {
#pragma unroll
    for (int i = 1; i < 16; ++i) tl[i] = 0;
    tl[0] = gtime();
  }
  const int R = a.B * a.Hkv;
  const int par_raw = __ldcg(a.parity);  // (in flight: first used when the predicted set is staged)
  const int ncl = gridDim.x / CS;
  bool waited = CS == 1;

#pragma unroll 1
  for (int it = 0, row = blockIdx.x / CS; row < R; ++it, row += ncl) {
    const uint32_t ipar = it & 1;  // phase of the once-per-row barriers
    const int b = row / a.Hkv, h = row - b * a.Hkv;
    const int len_ld = __ldcg(a.seq_lens + b);  // in flight; first USED below, after the requests that do not need it
    // The row's blocks are dealt to the CTAs by the STATIC bound NBH >= ceil(len / bs) (the caller's
    // max_blocks_per_seq or hint), so the summary requests go out without waiting for the length; rows
    // past the last block are fetched but never scored.
    const int nb4 = (a.NBH + 3) & ~3;
    const int slice = ((nb4 + CS - 1) / CS + 3) & ~3;
    const int s0 = min(nb4, (int)rank * slice), s1 = min(nb4, s0 + slice);
    const int nrows = s1 - s0;                // rows of the summary buffer this CTA scores (multiple of 4)
    const int NCH = (nrows + CHR - 1) / CHR;  // ring positions taken by summary chunks
    const int pos0 = sh.ring_pos;             // ring position of chunk 0 (same in every thread: read after a barrier)
    const int ema_rank = CS - 1;
    const int HLmine = (int)rank < a.G ? (a.G - (int)rank + CS - 1) / CS : 0;  // query heads this CTA reduces
    const int n_spec = a.spec ? (a.Bud - (int)rank + CS - 1) / CS : 0;         // predicted slots dealt to this CTA
    const int UREP0 = (a.Bud + CS - 1) / CS;                                   // first repair descriptor
    const int NSUB = (a.bs + ST - 1) / ST;
    const size_t rowoff = (size_t)row * a.MB;
    // requests that do not depend on the length, all in flight together (each may be a TLB miss + HBM miss)
    uint4 qpre[4] = {};
    double th0 = 0.0, th1 = 0.0, th2 = 0.0;
    int n_old = 0;
    if (warp < SCW) {
      const uint16_t* qb = a.q + ((size_t)b * a.Hq + (size_t)h * a.G) * D + (lane % LPR) * 8;
#pragma unroll
      for (int e = 0; e < 4; ++e)
        if (e < a.G) qpre[e] = __ldg(reinterpret_cast<const uint4*>(qb + (size_t)e * D));
      th0 = a.theta[b * 3 + 0]; th1 = a.theta[b * 3 + 1]; th2 = a.theta[b * 3 + 2];
      n_old = a.n_state[row];
    }
    int ppre0[4] = {-1, -1, -1, -1}, ppre1[4] = {-1, -1, -1, -1};  // both prediction buffers: the parity is in flight too
    if (warp == LDW && a.spec) {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int j = e * 32 + lane;
        if (j < a.Bud) { ppre0[e] = __ldcg(a.P0 + (size_t)row * a.Bud + j); ppre1[e] = __ldcg(a.P1 + (size_t)row * a.Bud + j); }
      }
    }
    int pos = pos0, cnext = 0;
    auto buf_acquire = [&](int p) -> int {  // (loader lane 0) ring position p -> buffer, once its previous tenant is consumed
      const int bi = p % NBUF;
      if (p >= NBUF) { wait_bar(&sh.empty[bi], ((p / NBUF) - 1) & 1, err, 3); fence_proxy_async(); }
      return bi;
    };
    auto issue_chunk = [&](int c) {
      const int bi = buf_acquire(pos);
      const int rows = min(CHR, nrows - c * CHR);
      const int rows_ld = max(0, min(rows, a.MB - (s0 + c * CHR)));  // (stay inside the row of the summary buffer)
      const uint32_t bytes = (uint32_t)rows_ld * D * 2;
      mbar_expect_tx(&sh.fullV[bi], 0u);  // (both barriers of a buffer complete once per tenant)
      mbar_expect_tx(&sh.fullK[bi], bytes);
      if (bytes) bulk_load(ring + (size_t)bi * T::BYTES, a.summ + (rowoff + s0 + (size_t)c * CHR) * LPR, bytes, &sh.fullK[bi]);
      sh.pos_unit[bi] = -1;
      ++pos;
    };
    if (warp == LDW && lane == 0) {
      mbar_expect_tx(&sh.bar_keys, (uint32_t)nb4 * 4u);
      if ((int)rank == ema_rank) mbar_expect_tx(&sh.bar_pred, a.Bud > 0 ? (uint32_t)nb4 * 4u : 0u);
      else mbar_arrive(&sh.bar_pred);
      mbar_expect_tx(&sh.bar_red, (uint32_t)(CS * HLmine * SW * 4));
      for (; cnext < NCH && cnext < NBUF; ++cnext) issue_chunk(cnext);
      if (tl) tl[11] = gtime();
    }
    const int len = len_ld + a.app;
    const int nb = max(0, min(a.NBH, (len + a.bs - 1) / a.bs));
    const int ob = len > 0 ? (len - 1) / a.bs : -1;  // the open block
    if (tl && lane == 0 && warp == LDW) tl[10] = gtime();
    // (every remote store is preceded by the cluster barrier: all CTAs have initialised their mbarriers)

    // =========================================================================================
    MARK(100);
    if (warp == LDW) {
      // ---- loader warp: the barriers are armed and the first summary chunks requested (above); now the
      // predicted set is staged (list, bitmask, unit descriptors), then lane 0 feeds the ring until the row is done
      if (!waited) { cluster_wait(); waited = true; }
      // the predicted set P (a3 of the previous step): list, bitmask, this CTA's unit descriptors
      if (a.spec) {
        const int32_t* P = ((par_raw & 1) ? a.P1 : a.P0) + (size_t)row * a.Bud;
#pragma unroll 1
        for (int j0 = 0; j0 < a.Bud; j0 += 32) {
          const int j = j0 + lane;
          int blk = -1;
          if (j0 < 128) {
            const int e = j0 >> 5;
            const int v0 = e == 0 ? ppre0[0] : e == 1 ? ppre0[1] : e == 2 ? ppre0[2] : ppre0[3];
            const int v1 = e == 0 ? ppre1[0] : e == 1 ? ppre1[1] : e == 2 ? ppre1[2] : ppre1[3];
            blk = (par_raw & 1) ? v1 : v0;
          } else if (j < a.Bud) {
            blk = __ldcg(P + j);
          }
          if (blk >= nb) blk = -1;
          if (j < a.Bud) {
            plist[j] = blk;
            if (blk >= 0) atomicOr(&pmask[blk >> 5], 1u << (blk & 31));
            if (j % CS == (int)rank) {
              const int page = blk >= 0 ? __ldg(a.table + (size_t)b * a.MB + blk) : 0;
              units[j / CS] = make_int2(blk, page);
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) {
        __threadfence_block();
        sh.spec_ready = 1;
        if (tl) tl[12] = gtime();
        for (; cnext < NCH; ++cnext) issue_chunk(cnext);
        // The ring's producer.  Speculative units (a4) go out in order until A is known; from then on the
        // repair units (a6) go first -- they are the critical path -- and a predicted block that missed is
        // not requested at all (PRR_DROP with the cut).  A wait for a free buffer is left as soon as A
        // becomes known, so that the next buffer goes to a repair unit.
        int u_spec = 0, sub_spec = 0, i_rep = 0, sub_rep = 0, nrep = -1;
        const unsigned long long t0w = gtime();
        uint32_t itw = 0;
#pragma unroll 1
        for (;;) {
          if (nrep < 0 && sh.sel_done) {
            __threadfence_block();
            nrep = sh.n_rep;
            if (tl) { tl[13] = gtime(); tl[14] = nrep; }
          }
          int u = -1, sub = 0;
          bool rep = false;
          if (nrep >= 0 && i_rep < nrep) {
            u = UREP0 + i_rep; sub = sub_rep; rep = true;
          } else {
            while (u_spec < n_spec) {  // next speculative unit worth a request
              const int blk = units[u_spec].x;
              bool skip = blk < 0;
              if (!skip && nrep >= 0 && !a.retain) skip = sh.no_hits || (a.cut && !((amask[blk >> 5] >> (blk & 31)) & 1u));
              if (!skip) break;
              ++u_spec; sub_spec = 0;
            }
            if (u_spec < n_spec) { u = u_spec; sub = sub_spec; }
          }
          if (u < 0) {
            if (nrep >= 0) break;  // everything is out
            __nanosleep(64);       // only A is missing
            if ((++itw & 1023u) == 0 && (long long)(gtime() - t0w) > (long long)WAIT_NS) { wait_fail(err, 4); break; }
            continue;
          }
          const int2 d = units[u];
          const int valid = min(ST, len - d.x * a.bs - sub * ST);
          const bool last_sub = sub + 1 >= NSUB || min(ST, len - d.x * a.bs - (sub + 1) * ST) <= 0;
          if (valid > 0) {
            const int bi = pos % NBUF;
            if (pos >= NBUF) {  // the buffer's previous tenant must be consumed
              const uint32_t par = ((pos / NBUF) - 1) & 1;
              // (try_wait may suspend the thread for a system-dependent time: while A is still unknown the probe must
              // not block, or the repair units -- the critical path -- are issued late)
              bool free_ = nrep < 0 ? mbar_test_wait(&sh.empty[bi], par) : mbar_try_wait_cl(&sh.empty[bi], par);
              if (!free_ && nrep < 0) {  // keep an eye on A while waiting
                while (!(free_ = mbar_test_wait(&sh.empty[bi], par)) && !sh.sel_done)
                  if ((++itw & 1023u) == 0 && (long long)(gtime() - t0w) > (long long)WAIT_NS) { wait_fail(err, 3); break; }
                if (!free_) continue;  // A is known now: choose again
              } else if (!free_) {
                wait_bar(&sh.empty[bi], par, err, 3);
              }
              fence_proxy_async();
            }
            unsigned char* Ks = ring + (size_t)bi * T::BYTES;
            const int y = (d.y * a.Hkv + h) * a.bs + sub * ST;
            sh.pos_unit[bi] = u | (sub << 20) | (rep ? 0x40000000 : 0);
            if (tl && rep && tl[8] == 0) tl[8] = gtime();
            mbar_expect_tx(&sh.fullK[bi], T::HALF);
#pragma unroll
            for (int i = 0; i < T::NBOX; ++i) tma_load_2d(Ks + i * T::BOX_BYTES, &a.mapK, i * 64, y, &sh.fullK[bi]);
            mbar_expect_tx(&sh.fullV[bi], T::HALF);
#pragma unroll
            for (int i = 0; i < T::NBOX; ++i) tma_load_2d(Ks + T::HALF + i * T::BOX_BYTES, &a.mapV, i * 64, y, &sh.fullV[bi]);
            ++pos;
            __threadfence_block();
            sh.q_issued = pos;
          }
          if (rep) { if (last_sub || valid <= 0) { ++i_rep; sub_rep = 0; } else ++sub_rep; }
          else { if (last_sub || valid <= 0) { ++u_spec; sub_spec = 0; } else ++sub_spec; }
        }
        MARK(111);
        sh.q_total = pos;
        __threadfence_block();
        sh.q_final = 1;
        if (tl) tl[9] = gtime();
        MARK(112);
      }
      __syncwarp();
      if (lane == 0) sh.ring_pos = pos;  // (read by everyone after the row's last barrier)
    } else {
      if (warp < SCW) {
      // ---- a0 + a1 + a8: score the slice, chunk by chunk (warps 0 .. 7, RPW rows of a chunk each) -----
      const int sub = lane / LPR, l = lane % LPR;
      // the table entries of the slice, for group A's repair units (its own threads fill them)
      if (warp < GAW)
        for (int i = tid; i < nrows; i += GAW * 32) tslice[i] = s0 + i < nb ? __ldg(a.table + (size_t)b * a.MB + s0 + i) : 0;
      const bool own_ob = a.app && ob >= s0 && ob < s1;  // this CTA appends the new token
      double qs[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) qs[j] = 0.0;
      {
        const uint16_t* qb = a.q + ((size_t)b * a.Hq + (size_t)h * a.G) * D + l * 8;
#pragma unroll 1
        for (int g0 = 0; g0 < a.G; g0 += 4) {  // four query rows per batch of loads (zeros add nothing)
          uint4 t[4];
#pragma unroll
          for (int e = 0; e < 4; ++e)
            t[e] = g0 == 0 ? qpre[e]
                           : (g0 + e < a.G ? __ldg(reinterpret_cast<const uint4*>(qb + (size_t)(g0 + e) * D)) : make_uint4(0, 0, 0, 0));
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const uint32_t w[4] = {t[e].x, t[e].y, t[e].z, t[e].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              qs[2 * j] += (double)bf16_lo(w[j]);
              qs[2 * j + 1] += (double)bf16_hi(w[j]);
            }
          }
        }
      }
      const double alpha = th0, beta = th1, gamma = th2;
      const double oma = __dsub_rn(1.0, alpha), omb = __dsub_rn(1.0, beta);
      double* Lg = a.ema_l + rowoff;
      double* Vg = a.ema_v + rowoff;
      const uint32_t keys_a = smem_u32(keys), bk_a = smem_u32(&sh.bar_keys);
      const int w_lo = warp * RPW;  // this warp's first row inside a chunk
      if (!waited) { cluster_wait(); waited = true; }
#pragma unroll 1
      for (int c = 0; c < NCH; ++c) {
        const int p = pos0 + c, bi = p % NBUF;
        const int rows_c = min(CHR, nrows - c * CHR);  // (multiple of 4)
        const int g0r = s0 + c * CHR;                  // global block index of the chunk's row 0
        MARK(200 + c);
        if (tl && lane == 0 && c == 0) tl[14] = gtime();
        wait_bar(&sh.fullK[bi], (p / NBUF) & 1, err, 5);
        if (tl && lane == 0 && c == 0) tl[6] = gtime();
        if (tl && lane == 0 && c == 1 && warp >= 4) tl[12] = gtime();
        uint4* st = reinterpret_cast<uint4*>(ring + (size_t)bi * T::BYTES);
        if (own_ob && ob >= g0r + w_lo && ob < g0r + min(rows_c, w_lo + RPW)) {
          // a0: the block the new token falls in is scored after the append: its summary row was computed
          // by a tile warp while the chunk was in flight (below); patch the staged row
          if (lane == 0) wait_flag(&sh.patch_ready, err, 15);
          __syncwarp();
          __threadfence_block();
          if (sub == 0) st[(ob - g0r) * LPR + l] = *reinterpret_cast<const uint4*>(&sh.patch_row[l * 4]);
          __syncwarp();
        }
        // Exact dot products (Q1): every partial sum is exact in fp64, so the order is free.  Lane group
        // `sub` takes the rows w_lo + e RW + sub, e < NV, all requested and converted before the first
        // shuffle; the NV partial sums per lane are folded across the LPR lanes by a transposed butterfly
        // (each step halves what a lane carries), then a plain butterfly over the remaining lanes.
        if (w_lo < rows_c) {  // (warp-uniform)
        double acc[NV];
#pragma unroll
        for (int e = 0; e < NV; ++e) {
          const int r = w_lo + e * RW + sub;
          const uint4 v = r < rows_c ? st[r * LPR + l] : make_uint4(0, 0, 0, 0);
          const uint32_t w[4] = {v.x, v.y, v.z, v.w};
          double a0 = 0.0, a1 = 0.0;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            a0 = fma((double)bf16_lo(w[j]), qs[2 * j], a0);
            a1 = fma((double)bf16_hi(w[j]), qs[2 * j + 1], a1);
          }
          acc[e] = a0 + a1;
        }
        int eidx = 0;
        {
          int off = LPR / 2;
#pragma unroll
          for (int nvv = NV; nvv > 1; nvv >>= 1, off >>= 1) {
            const bool up = (l & off) != 0;
#pragma unroll
            for (int j = 0; j < nvv / 2; ++j)
              acc[j] = (up ? acc[nvv / 2 + j] : acc[j]) + __shfl_xor_sync(FULL, up ? acc[j] : acc[nvv / 2 + j], off);
            eidx += up ? nvv / 2 : 0;
          }
#pragma unroll
          for (; off >= 1; off >>= 1) acc[0] += __shfl_xor_sync(FULL, acc[0], off);
        }
        {
          const int r = w_lo + eidx * RW + sub;
          if ((l & (LPR / NV - 1)) == 0 && r < rows_c)
            scs[c * CHR + r] = g0r + r < nb ? f64_to_score(__dmul_rn(acc[0], a.score_c)) : 0.f;
        }
        }
        __syncwarp();
        if (tl && lane == 0 && warp >= 4 && c < 2) tl[c == 0 ? 10 : 13] = gtime();
        // this warp is done with the buffer
        if (lane == 0) {
          const int old = atomicAdd(&sh.chunk_cnt[bi], 1);
          if (old == SCW - 1) { sh.chunk_cnt[bi] = 0; mbar_arrive(&sh.empty[bi]); }
        }
        // keys out: one st.async of four consecutive keys per (group of four rows, destination CTA) pair,
        // one pair per lane
        uint32_t key = 0u;
        if (lane < RPW && w_lo + lane < rows_c) {
          const int i = g0r + w_lo + lane;
          if (i < nb) {
            const float sv = scs[c * CHR + w_lo + lane];
            a.scores[rowoff + i] = sv;
            key = score_key(sv);
          }
        }
        {
          constexpr int NGRP = RPW / 4;
#pragma unroll 1
          for (int pi0 = 0; pi0 < NGRP * CS; pi0 += 32) {
            const int pi = pi0 + lane;
            const int grp = min(pi / CS, NGRP - 1), dest = pi % CS;
            const uint32_t k0 = __shfl_sync(FULL, key, 4 * grp), k1 = __shfl_sync(FULL, key, 4 * grp + 1);
            const uint32_t k2 = __shfl_sync(FULL, key, 4 * grp + 2), k3 = __shfl_sync(FULL, key, 4 * grp + 3);
            if (pi < NGRP * CS && w_lo + 4 * grp < rows_c) {
              const uint32_t off = (uint32_t)(g0r + w_lo + 4 * grp) * 4u;
              st_async_v4(mapa(keys_a + off, dest), k0, k1, k2, k3, mapa(bk_a, dest));
            }
          }
        }
        if (tl && lane == 0 && warp >= 4 && c == 0) tl[11] = gtime();
      }
      if (tl && lane == 0) tl[1] = gtime();
      MARK(300);
      }  // scoring warps
      if (!waited) { cluster_wait(); waited = true; }
      // ---- a2: the true top-K (keys in registers, no histogram) when the row fits the fast path
      const int kA = min(a.K, nb);
      const bool fastA = nb <= 256 * 18 && kA <= 256;
      if (warp < SCW && fastA) {
        const Grp g4{tid, SCW * 32, warp, SCW, 1};
        const SelMem m4{hist, red, cand, offs};
        MARK(700);
        wait_bar(&sh.bar_keys, ipar, err, 9);  // every CTA's keys have landed
        MARK(701);
        if (tl && lane == 0) tl[7] = gtime();
        if (nb <= 256 * 9) grp_select_v3<256, 9>(keys, nb, kA, g4, m4, amask, tl);
        else grp_select_v3<256, 18>(keys, nb, kA, g4, m4, amask, tl);
        g4.sync();
        if (tl && lane == 0) tl[8] = gtime();
      }

      // =======================================================================================
      if (warp == 10 && a.app && ob >= s0 && ob < s1) {
        // a0 by an idle tile warp, off the scoring warps' critical path: cache slot, running sum and mean-key
        // summary of the open block (exact fp64 sum, one division, one RNE to bf16, Q2), D / 32 channels per lane
        constexpr int CPL = D / 32;  // 2 or 4 channels = 1 or 2 words per lane
        const int pos_t = len - 1, slot = pos_t - ob * a.bs;
        const size_t ch = ((size_t)b * a.Hkv + h) * D + lane * CPL;
        const size_t page = (size_t)__ldg(a.table + (size_t)b * a.MB + ob);
        const size_t dst = ((page * a.Hkv + h) * a.bs + slot) * (size_t)D + lane * CPL;
        uint32_t kw[CPL / 2], vw[CPL / 2], o[CPL / 2];
#pragma unroll
        for (int j = 0; j < CPL / 2; ++j) {
          kw[j] = __ldg(reinterpret_cast<const uint32_t*>(a.k_new + ch) + j);
          vw[j] = __ldg(reinterpret_cast<const uint32_t*>(a.v_new + ch) + j);
        }
        double s_old[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) s_old[j] = slot == 0 ? 0.0 : a.open_sum[ch + j];
#pragma unroll
        for (int j = 0; j < CPL / 2; ++j) {
          reinterpret_cast<uint32_t*>(a.kp_w + dst)[j] = kw[j];
          reinterpret_cast<uint32_t*>(a.vp_w + dst)[j] = vw[j];
          const double x0 = (double)bf16_lo(kw[j]), x1 = (double)bf16_hi(kw[j]);
          const double a0 = slot == 0 ? x0 : __dadd_rn(s_old[2 * j], x0);
          const double a1 = slot == 0 ? x1 : __dadd_rn(s_old[2 * j + 1], x1);
          a.open_sum[ch + 2 * j] = a0;
          a.open_sum[ch + 2 * j + 1] = a1;
          o[j] = (uint32_t)f64_to_bf16_rne(__ddiv_rn(a0, (double)(slot + 1))) |
                 ((uint32_t)f64_to_bf16_rne(__ddiv_rn(a1, (double)(slot + 1))) << 16);
          sh.patch_row[lane * (CPL / 2) + j] = o[j];
          reinterpret_cast<uint32_t*>(a.summ_w + (rowoff + ob) * LPR)[lane * (CPL / 2) + j] = o[j];
        }
        __syncwarp();
        if (lane == 0) { __threadfence_block(); sh.patch_ready = 1; }
      }
      if (warp >= TW0) {
        {
        // ---- tile warps: a4 + a6.  Ring positions are claimed in order; a speculative partial whose
        // fate is unknown is parked in a slot, everything else is folded into this warp's running state.
        float* wst = slots + (size_t)(a.NSLOT + warp - TW0) * SLOTF;
        const float sl2 = a.scale * LOG2E_F;
        const int NG = (a.G + 7) >> 3;
        uint32_t qb[D / 16][2];  // query fragments of pass `qps` (one pass unless G > 8: then reloaded, from L1)
        int qps = -1;
        auto load_q = [&](int ps) {
          const uint16_t* qg = a.q + ((size_t)b * a.Hq + (size_t)h * a.G) * D;
          const int g = ps * 8 + (lane >> 2), tq = lane & 3;
#pragma unroll
          for (int k16 = 0; k16 < D / 16; ++k16) {
            const int col = k16 * 16 + tq * 2;
            qb[k16][0] = g < a.G ? __ldg(reinterpret_cast<const uint32_t*>(qg + g * D + col)) : 0u;
            qb[k16][1] = g < a.G ? __ldg(reinterpret_cast<const uint32_t*>(qg + g * D + col + 8)) : 0u;
          }
          qps = ps;
        };
        load_q(0);
        // running state of the first eight query heads in REGISTERS (Eq. 6-8, unnormalised, m in log2 units);
        // further heads (G > 8, second pass) fold into the shared-memory image
        float orun[D / 16][4], mrun[2] = {-CUDART_INF_F, -CUDART_INF_F}, lrun[2] = {0.f, 0.f};
#pragma unroll
        for (int dt = 0; dt < D / 16; ++dt)
#pragma unroll
          for (int e = 0; e < 4; ++e) orun[dt][e] = 0.f;
#pragma unroll 1
        for (;;) {
          int p = 0;
          if (lane == 0) p = pos0 + NCH + atomicAdd(&sh.t_next, 1);  // tile positions follow the row's chunks
          p = __shfl_sync(FULL, p, 0);
          bool done = false;
          MARK(400 + (p & 63));
          if (lane == 0) {  // wait until position p is in flight, or the queue is final and shorter
            const unsigned long long t0 = gtime();
            uint32_t itw = 0;
            for (;;) {
              if (p < sh.q_issued) break;
              if (sh.q_final) { __threadfence_block(); if (p >= sh.q_total) { done = true; } break; }
              __nanosleep(32);
              if ((++itw & 1023u) == 0 && (long long)(gtime() - t0) > (long long)WAIT_NS) { wait_fail(err, 14); done = true; break; }
            }
          }
          done = __shfl_sync(FULL, (int)done, 0) != 0;
          if (done) break;
          __threadfence_block();
          const int bi = p % NBUF;
          const uint32_t par = (p / NBUF) & 1;
          const int pu = sh.pos_unit[bi];
          const bool rep = (pu & 0x40000000) != 0;
          const int u = pu & 0xfffff, sub_t = (pu >> 20) & 0x3ff;
          const int2 d = units[u];
          const int blk = d.x;
          const int valid = min(ST, len - blk * a.bs - sub_t * ST);
          unsigned char* Ks = ring + (size_t)bi * T::BYTES;
          const bool patch = a.app && blk == ob && (len - 1 - ob * a.bs) / ST == sub_t;
          const uint16_t* pk = patch ? a.k_new + ((size_t)b * a.Hkv + h) * D : nullptr;
          const uint16_t* pv = patch ? a.v_new + ((size_t)b * a.Hkv + h) * D : nullptr;
          // fate of a speculative unit: 1 merge, 0 drop, -1 unknown (park)
          // (read by ONE lane and broadcast: the flag may flip between two lanes' reads, and the warp
          // must take one path through the warp-synchronous tile code)
          auto fate = [&]() -> int {
            if (rep || a.retain) return 1;
            int f = -1;
            if (lane == 0 && sh.sel_done) {
              __threadfence_block();
              f = sh.no_hits ? 0 : (int)((amask[blk >> 5] >> (blk & 31)) & 1u);
            }
            return __shfl_sync(FULL, f, 0);
          };
          MARK(500 + (p & 63));
          const unsigned long long tc0 = tl ? gtime() : 0ull;
          if (tl && lane == 0) { tl[13] += 1; if (rep && tl[10] == 0) tl[10] = tc0; }
          int f = fate();
          if (f == 0) {  // already known to be over-predicted: let the tile land, free the buffer
            wait_bar(&sh.fullK[bi], par, err, 6);
            wait_bar(&sh.fullV[bi], par, err, 7);
            __syncwarp();
            if (lane == 0) mbar_arrive(&sh.empty[bi]);
            continue;
          }
          float* dst = wst;
          bool fold = true;
          int slot = -1;
          unsigned long long tcw = 0ull;
          if (tl) { wait_bar(&sh.fullK[bi], par, err, 6); tcw = gtime(); }
#pragma unroll 1
          for (int ps = 0; ps < NG; ++ps) {  // (one copy of the tile code: the instruction cache is small)
            if (ps != qps) load_q(ps);
            float o[D / 16][4], mt[2], lt[2];
            const unsigned long long tp0 = tl ? gtime() : 0ull;
            tile_partial<D, ST>(Ks, &sh.fullK[bi], &sh.fullV[bi], par, qb, valid, sl2, pk, pv, ps == 0, o, mt, lt, err, warp >= 8 ? tl : nullptr);
            if (tl && lane == 0 && warp >= 8) { tl[6] += tl[1] - tp0; tl[3] = gtime(); }
            if (ps == NG - 1) {  // every lane is done with the tile: the buffer may be refilled
              __syncwarp();
              if (lane == 0) mbar_arrive(&sh.empty[bi]);
            }
            if (ps == 0) {
              f = fate();
              if (f < 0) {  // park it, if a slot is left; else wait for A
                if (lane == 0) slot = atomicAdd(&sh.n_slots, 1);
                slot = __shfl_sync(FULL, slot, 0);
                if (slot < a.NSLOT) {
                  dst = slots + (size_t)slot * SLOTF;
                  fold = false;
                  if (lane == 0) slotblk[slot] = blk | (sub_t << 20);
                } else {
                  if (lane == 0) wait_flag(&sh.sel_done, err, 8);
                  __syncwarp();
                  f = fate();
                }
              }
            }
            if (f != 0) {
              if (fold && ps == 0) {
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                  const float mn = fmaxf(mrun[j], mt[j]);
                  const float al = mrun[j] == -CUDART_INF_F ? 0.f : ex2(mrun[j] - mn), be = ex2(mt[j] - mn);
                  lrun[j] = al * lrun[j] + be * lt[j];
                  mrun[j] = mn;
#pragma unroll
                  for (int dt = 0; dt < D / 16; ++dt) {
                    orun[dt][j] = al * orun[dt][j] + be * o[dt][j];
                    orun[dt][2 + j] = al * orun[dt][2 + j] + be * o[dt][2 + j];
                  }
                }
              } else {
                state_put<D>(dst, a.G, ps, o, mt, lt, fold);
              }
            }
            if (tl && lane == 0 && warp >= 8) tl[7] += gtime() - tl[3];
          }
          if (tl && lane == 0) {
            const unsigned long long tc1 = gtime();
            if (rep && tl[12] == 0) tl[12] = tc1;
            tl[14] += tc1 - tc0;                      // total time in tiles (wait for the data + compute)
            tl[8] += tcw - tc0;                       // ... of which waiting for K
            if (tl[11] == 0) tl[11] = tc1 - tc0;      // first tile
            tl[9] = tc1 - tc0;                        // last tile
          }
        }
        state_put<D>(wst, a.G, 0, orun, mrun, lrun, false);  // the running state, for the merge
        __syncwarp();
        if (lane == 0) mbar_arrive(&sh.bar_tw);
        MARK(600);
        if (tl && lane == 0) tl[4] = gtime();
        }
      } else if (warp < GA0 + GAW) {
        // ---- group A: true top-K (a2), diff (a5), repair units, lists, merge (a7) ----------------------
        const Grp g{tid - GA0 * 32, GAW * 32, warp - GA0, GAW, 2};
        const SelMem m{hist, red, cand, offs};
        if (!fastA) {  // long rows or K > 256: the generic narrowing, by this group alone
          MARK(700);
          wait_bar(&sh.bar_keys, ipar, err, 9);
          MARK(701);
          if (tl && lane == 0) tl[7] = gtime();
          Thr t;
          t.key = 0u; t.idx = 0x7fffffff;  // k >= n: everything is selected
          if (kA < nb) t = grp_kth(keys, nb, kA, g, m, tl);
          grp_mask(keys, nb, kA, t, g, amask);
          if (tl && lane == 0) tl[8] = gtime();
        }
        if (g.tid == 0) wait_flag(&sh.spec_ready, err, 10);
        g.sync();
        // repair units: the missed blocks of this CTA's slice (all of A's in the sequential path)
        bool all_rep = false;
        if (a.recompute && !a.retain) {  // S1: does the row have a miss at all?  (every CTA holds the whole bitmasks)
          int mc = 0;
          for (int w = g.tid; w < (nb + 31) >> 5; w += g.nt) mc += __popc(amask[w] & ~pmask[w]);
          mc = __reduce_add_sync(FULL, mc);
          if (lane == 0 && mc) atomicAdd(&sh.miss_cnt, mc);
          g.sync();
          all_rep = sh.miss_cnt > 0;
        }
        {  // one shared-memory atomic per warp and trip (same-address atomics serialise: 64 of them cost ~1 us)
          const int lim = min(s1, nb);
#pragma unroll 1
          for (int i0 = s0 + g.wid * 32; i0 < lim; i0 += g.nt) {
            const int i = i0 + lane;
            const uint32_t bit = 1u << (i & 31);
            const bool rep_i = i < lim && (amask[i >> 5] & bit) && (all_rep || !(pmask[i >> 5] & bit));
            const uint32_t bal = __ballot_sync(FULL, rep_i);
            int base = 0;
            if (lane == 0 && bal) base = atomicAdd(&sh.rep_cnt, __popc(bal));
            base = __shfl_sync(FULL, base, 0);
            if (rep_i) units[UREP0 + base + __popc(bal & ((1u << lane) - 1u))] = make_int2(i, tslice[i - s0]);
          }
        }
        g.sync();
        if (g.tid == 0) {
          sh.n_rep = sh.rep_cnt;
          sh.no_hits = all_rep ? 1 : 0;
          __threadfence_block();
          sh.sel_done = 1;
        }
        if (tl && lane == 0) tl[2] = gtime();
        // a8 (Eq. 3) and the prediction for the next step (Eq. 2), off the critical path: the slice's scores are
        // in shared memory; four consecutive blocks per thread (one st.async of prediction keys)
        {
          const uint32_t pkeys_a = smem_u32(pkeys), bp_a = smem_u32(&sh.bar_pred);
          const double alpha = th0, beta = th1, gamma = th2;
          const double oma = __dsub_rn(1.0, alpha), omb = __dsub_rn(1.0, beta);
          double* Lg = a.ema_l + rowoff;
          double* Vg = a.ema_v + rowoff;
#pragma unroll 1
          for (int r4 = g.tid * 4; r4 < nrows; r4 += g.nt * 4) {
            double el[4], ev[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int i = s0 + r4 + e;
              const bool has = i < min(nb, n_old);
              el[e] = has ? Lg[i] : 0.0;
              ev[e] = has ? Vg[i] : 0.0;
            }
            uint32_t pk[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int i = s0 + r4 + e;
              pk[e] = 0u;
              if (i < nb) {
                const double xd = (double)scs[r4 + e];
                double ln = xd, vn = 0.0;
                if (i < n_old) {  // non-contracted fp64, both lines use l^{t-1} (Q5)
                  vn = __dadd_rn(__dmul_rn(beta, __dsub_rn(xd, el[e])), __dmul_rn(omb, ev[e]));
                  ln = __dadd_rn(__dmul_rn(alpha, xd), __dmul_rn(oma, el[e]));
                }
                Lg[i] = ln;
                Vg[i] = vn;
                pk[e] = score_key(f64_to_score(__dadd_rn(ln, __dmul_rn(gamma, vn))));
              }
            }
            if (a.Bud > 0) st_async_v4(mapa(pkeys_a + (uint32_t)(s0 + r4) * 4u, ema_rank), pk[0], pk[1], pk[2], pk[3], mapa(bp_a, ema_rank));
          }
        }
        if (rank == 0) {  // the row's lists as the API reports them, off the critical path
          const uint32_t tot = grp_emit(amask, pmask, nb, g, m, a.setA + (size_t)row * a.K, a.K,
                                        a.setM + (size_t)row * a.K, a.K);
          if (g.tid == 0) {
            int np = 0;
            for (int j = 0; j < (a.spec ? a.Bud : 0); ++j) np += plist[j] >= 0;
            const int nA = (int)(tot >> 16), nM = (int)(tot & 0xffffu);
            a.counts[row * 3 + 0] = nA;
            a.counts[row * 3 + 1] = np;
            a.counts[row * 3 + 2] = nM;
            a.n_state[row] = nb;
            if (a.stats) {
              atomicAdd(&a.stats[0], (unsigned long long)nA);
              atomicAdd(&a.stats[1], (unsigned long long)(nA - nM));
              atomicAdd(&a.stats[2], (unsigned long long)nM);
              atomicAdd(&a.stats[3], (unsigned long long)np);
            }
          }
        }
        if ((int)rank == ema_rank && a.Bud > 0) {
          // ---- P of the next step = top-min(Bud, #stateful) of the Eq. 2 predictions (a3), on one CTA of the
          // cluster, by the same group with the same code, while the repair tiles are in flight
          uint32_t* emask = offs + 2 * a.MBw;  // [MBw]
          MARK(800);
          wait_bar(&sh.bar_pred, ipar, err, 13);
          MARK(801);
          const int bsel = a.bud_seq[b] > 0 ? min(a.bud_seq[b] - 1, a.Bud) : a.BudSel;
          const int kp = min(bsel, nb);
          if (kp == 0) {
            for (int w = g.tid; w < a.MBw; w += g.nt) emask[w] = 0u;
          } else if (nb <= 128 * 18 && kp <= 128) {
            grp_select_v3<128, 18>(pkeys, nb, kp, g, m, emask, nullptr);
          } else if (nb <= 128 * 36 && kp <= 128) {
            grp_select_v3<128, 36>(pkeys, nb, kp, g, m, emask, nullptr);
          } else {
            Thr tp;
            tp.key = 0u; tp.idx = 0x7fffffff;
            if (kp < nb) tp = grp_kth(pkeys, nb, kp, g, m);
            grp_mask(pkeys, nb, kp, tp, g, emask);
          }
          g.sync();
          grp_emit(emask, nullptr, nb, g, m, ((par_raw & 1) ? a.P0 : a.P1) + (size_t)row * a.Bud, a.Bud, nullptr, 0);
          if (tl && lane == 0) tl[9] = gtime();
        }
        // ---- merge: this CTA's hit slots and warp states per query head, then to the head's reducer
        MARK(710);
        wait_bar(&sh.bar_tw, ipar, err, 11);
        MARK(711);
        __threadfence_block();
        if (tl && lane == 0) tl[3] = gtime();
        const int nsl = min(sh.n_slots, a.NSLOT);
        const uint32_t recv_a = smem_u32(recv), br_a = smem_u32(&sh.bar_red);
#pragma unroll 1
        for (int gq = g.wid; gq < a.G; gq += GAW) {
          float mrun = -CUDART_INF_F, lrun = 0.f;
          float4 acc[D / 128 > 0 ? D / 128 : 1];
          constexpr int NV = D / 128 > 0 ? D / 128 : 1;
          const bool on = lane * 4 < D;
#pragma unroll
          for (int v = 0; v < NV; ++v) acc[v] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
          for (int e = 0; e < nsl + NTW; ++e) {
            if (e < nsl) {
              const int blk = slotblk[e] & 0xfffff;
              if (!a.retain && (sh.no_hits || !((amask[blk >> 5] >> (blk & 31)) & 1u))) continue;
            }
            const float* st = slots + (size_t)(e < nsl ? e : a.NSLOT + (e - nsl)) * SLOTF + gq * SW;
            const float me = st[0], le = st[1];
            if (me == -CUDART_INF_F) continue;
            const float mn = fmaxf(mrun, me);
            const float fo = mrun == -CUDART_INF_F ? 0.f : ex2(mrun - mn), fn = ex2(me - mn);
            lrun = fo * lrun + fn * le;
            mrun = mn;
#pragma unroll
            for (int v = 0; v < NV; ++v) {
              const float4 x = on ? *reinterpret_cast<const float4*>(st + 4 + v * 128 + lane * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
              acc[v].x = fo * acc[v].x + fn * x.x; acc[v].y = fo * acc[v].y + fn * x.y;
              acc[v].z = fo * acc[v].z + fn * x.z; acc[v].w = fo * acc[v].w + fn * x.w;
            }
          }
          const int rr = gq % CS, hl = gq / CS;
          const uint32_t dsta = recv_a + (uint32_t)((rank * a.HL + hl) * SW) * 4u;
          const uint32_t ra = CS > 1 ? mapa(dsta, rr) : dsta, rb = CS > 1 ? mapa(br_a, rr) : br_a;
          if (lane == 0) st_async_v4(ra, __float_as_uint(mrun), __float_as_uint(lrun), 0u, 0u, rb);
#pragma unroll
          for (int v = 0; v < NV; ++v)
            if (on) st_async_v4(ra + 16u + (uint32_t)(v * 128 + lane * 4) * 4u, __float_as_uint(acc[v].x), __float_as_uint(acc[v].y),
                                __float_as_uint(acc[v].z), __float_as_uint(acc[v].w), rb);
        }
        // ---- reducer: fold the cluster's partials of this CTA's query heads, normalise, write out
        if (HLmine > 0) {
          MARK(720);
          wait_bar(&sh.bar_red, ipar, err, 12);
          MARK(721);
#pragma unroll 1
          for (int hl = g.wid; hl < HLmine; hl += GAW) {
            const int gq = hl * CS + (int)rank;
            constexpr int NV = D / 128 > 0 ? D / 128 : 1;
            const bool on = lane * 4 < D;
            float mrun = -CUDART_INF_F, lrun = 0.f;
            float4 acc[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) acc[v] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
            for (int r = 0; r < CS; ++r) {
              const float* st = recv + (size_t)(r * a.HL + hl) * SW;
              const float me = st[0], le = st[1];
              if (me == -CUDART_INF_F) continue;
              const float mn = fmaxf(mrun, me);
              const float fo = mrun == -CUDART_INF_F ? 0.f : ex2(mrun - mn), fn = ex2(me - mn);
              lrun = fo * lrun + fn * le;
              mrun = mn;
#pragma unroll
              for (int v = 0; v < NV; ++v) {
                const float4 x = on ? *reinterpret_cast<const float4*>(st + 4 + v * 128 + lane * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
                acc[v].x = fo * acc[v].x + fn * x.x; acc[v].y = fo * acc[v].y + fn * x.y;
                acc[v].z = fo * acc[v].z + fn * x.z; acc[v].w = fo * acc[v].w + fn * x.w;
              }
            }
            const float inv = lrun > 0.f ? 1.f / lrun : 0.f;
            float* op = a.out + ((size_t)b * a.Hq + (size_t)h * a.G + gq) * D;
#pragma unroll
            for (int v = 0; v < NV; ++v)
              if (on) *reinterpret_cast<float4*>(op + v * 128 + lane * 4) =
                  make_float4(acc[v].x * inv, acc[v].y * inv, acc[v].z * inv, acc[v].w * inv);
          }
        }
        if (tl && lane == 0) tl[5] = gtime();
      }
    }
    MARK(900);
    __syncthreads();  // the row is done in this CTA
    MARK(901);
    if (row + ncl < R) {  // (one CTA per row and more rows than CTAs)
      row_init();
      __syncthreads();
    }
    if (tl && lane == 0 && tl[5] == 0) tl[5] = gtime();
  }
  if (!waited) cluster_wait();
  if (CS > 1) {  // nobody leaves while a peer may still be storing into the cluster's shared memory
    cluster_arrive();
    cluster_wait();
    MARK(902);
  }

  if (tl && lane < 15) tlg[lane] = tl[lane];
  // ---- exit: the last CTA of the grid flips the parity and bumps the lengths -------------------
  if (tid == 0) {
    __threadfence();
    const uint32_t last = atomicAdd(&a.ctl[CTL_EXIT], 1u) == gridDim.x - 1 ? 1u : 0u;
    if (last && a.done_host) {
      __threadfence_system();
      *reinterpret_cast<volatile uint32_t*>(a.done_host) = a.done_seq;
    }
    if (last) {
      a.ctl[CTL_EXIT] = 0u;
      *a.parity = par_raw ^ 1;
      if (a.app)
        for (int b = 0; b < a.B; ++b)
          if (a.seq_lens_w[b] / a.bs < a.MB) a.seq_lens_w[b] += 1;  // (a full sequence: nothing was written, the length stays, as in k_append)
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
struct RowPlan { int CS, NBUF, NSLOT, smem; };

template <int D, int ST>
static cudaError_t plan_and_launch(prr_ctx* c, RowArgs& a, cudaStream_t s) {
  using T = Tile<D, ST>;
  const int R = a.B * a.Hkv;
  const void* fn = (const void*)k_row<D, ST>;
  const int key = (D == 128 ? 0 : 1) * 3 + (ST == 64 ? 0 : ST == 32 ? 1 : 2);
  if (!c->row_attr[key]) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return e;
    c->row_dyn[key] = c->smem_optin - (int)fa.sharedSizeBytes;
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, c->row_dyn[key]);
    if (e != cudaSuccess) return e;
    // clusters of 1, 2, 4, 8, 16 CTAs that can be co-resident with the whole shared memory of an SM each
    // (16 is past the portable size: the function opts in)
    const bool np16 = cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
    if (!np16) cudaGetLastError();
    for (int i = 0; i < 5; ++i) {
      if (i == 4 && !np16) { c->row_maxcl[key][i] = 0; continue; }
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((1 << i) * 8); cfg.blockDim = dim3(NTHR);
      cfg.dynamicSmemBytes = c->row_dyn[key];
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = 1 << i; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      int n = 0;
      if (cudaOccupancyMaxActiveClusters(&n, fn, &cfg) != cudaSuccess) { cudaGetLastError(); n = i == 0 ? c->n_sm : 0; }
      c->row_maxcl[key][i] = n;
    }
    c->row_attr[key] = 1;
  }
  // the largest cluster that still gives every row its own cluster in one wave
  int CS = 1;
  for (int i = 4; i >= 0; --i)
    if (c->row_maxcl[key][i] >= R) { CS = 1 << i; break; }
  if (c->force_cs > 0) CS = c->force_cs;
  int li = 0; while ((1 << li) < CS) ++li;
  const int ncl = std::max(1, std::min(R, c->row_maxcl[key][li] > 0 ? c->row_maxcl[key][li] : 1));
  if (CS > 1 && ncl < R) return cudaErrorInvalidConfiguration;
  a.CS = CS;
  a.HL = (a.G + CS - 1) / CS;
  a.UCAP = (a.Bud + CS - 1) / CS + a.K;  // (S1 makes every block of A in the slice a repair unit: <= K)
  a.SLMAX = ((((a.MB + 3) & ~3) + CS - 1) / CS + 3 + 4) & ~3;
  const int SW = D + 4, SLOTF = a.G * SW;
  // a slot per speculative unit of a CTA if they fit (a unit whose fate is unknown and that finds no slot
  // holds its warp until A is known); then the deepest ring; a ring of at least four tenants comes first
  // (the sequential path parks nothing: its shared memory goes to the ring)
  // (and a small run-time budget parks few: a.BudMax is the largest budget in force among the launch's sequences)
  a.NSLOT = a.spec ? std::max(1, std::min(16, ((std::min(a.Bud, a.BudMax) + CS - 1) / CS) * ((a.bs + ST - 1) / ST))) : 1;
  const int min_ring = 4;
  const int budget = c->row_dyn[key];
  int NBUF = NBMAX;
  for (;;) {
    int o = NBUF * T::BYTES;
    auto take = [&](int bytes) { const int at = o; o += (bytes + 15) & ~15; return at; };
    a.o_keys = take((a.MB + 8) * 4);
    a.o_pkeys = take((a.MB + 8) * 4);
    a.o_hist = take(2 * HB * 4);
    a.o_plist = take(std::max(1, a.Bud) * 4);
    a.o_pmask = take(a.MBw * 4);
    a.o_amask = take(a.MBw * 4);
    a.o_offs = take(3 * a.MBw * 4);  // emission offsets (2 groups) + the prediction bitmask
    a.o_tslice = take(a.SLMAX * 4);
    a.o_sc = take(a.SLMAX * 4);
    a.o_units = take(a.UCAP * 8);
    a.o_cand = take((CANDX + 64) * 8);
    a.o_red = take(2 * 32 * 4);
    a.o_slots = take((a.NSLOT + NTW) * SLOTF * 4);
    a.o_slotblk = take(a.NSLOT * 4);
    a.o_recv = take(CS * a.HL * SW * 4);
    a.o_end = o;
    if (o <= budget) break;
    if (NBUF > min_ring) { --NBUF; continue; }
    if (a.NSLOT > 1) { --a.NSLOT; continue; }
    if (NBUF > 1) { --NBUF; continue; }
    return cudaErrorInvalidConfiguration;
  }
  a.NBUF = NBUF;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(ncl * CS);
  cfg.blockDim = dim3(NTHR);
  cfg.dynamicSmemBytes = a.o_end;
  cfg.stream = s;
  cudaLaunchAttribute at[2];
  int na = 0;
  {  // (also for one CTA per row: st.async needs a cluster launch)
    at[na].id = cudaLaunchAttributeClusterDimension;
    at[na].val.clusterDim.x = CS; at[na].val.clusterDim.y = 1; at[na].val.clusterDim.z = 1;
    ++na;
  }
  if (c->pdl) {
    at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
  }
  cfg.attrs = at; cfg.numAttrs = na;
  c->last_cs = CS; c->last_nbuf = NBUF; c->last_grid = ncl * CS;
  return cudaLaunchKernelEx(&cfg, k_row<D, ST>, a);
}

// Tensor map of a K or V page pool for the copy engine: bf16 [rows, d] with rows = page * Hkv * bs
// (the library is not told n_pages; tile coordinates are int32, so the row extent is 2^31), box =
// [ST rows, 64 channels = 128 bytes], 128-byte swizzle.  Encoded on the host, cached per pointer.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess) p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}
static int page_map(prr_ctx* c, const void* base, int box_rows, CUtensorMap* out) {
  static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap is 128 bytes");
  const void* key = reinterpret_cast<const void*>(reinterpret_cast<uintptr_t>(base) | (uintptr_t)(box_rows / 16 - 1));  // (16-byte aligned base)
  auto it = c->tmaps.find(key);
  if (it == c->tmaps.end()) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return (int)cudaErrorNotSupported;
    alignas(64) CUtensorMap m;
    const cuuint64_t dims[2] = {(cuuint64_t)c->D, (cuuint64_t)1 << 31};
    const cuuint64_t strides[1] = {(cuuint64_t)c->D * 2};
    const cuuint32_t box[2] = {64u, (cuuint32_t)box_rows};
    const cuuint32_t es[2] = {1u, 1u};
    if (fn(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, es,
           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return (int)cudaErrorInvalidValue;
    std::array<uint64_t, 16> blob;
    memcpy(blob.data(), &m, 128);
    if (c->tmaps.size() > 4096) c->tmaps.clear();
    it = c->tmaps.emplace(key, blob).first;
  }
  memcpy(out, it->second.data(), 128);
  return 0;
}

}  // namespace cluster
using namespace cluster;

int launch_step_cluster(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries, float* out,
                        int spec, cudaStream_t s, const void* k_new, const void* v_new) {
  const size_t r = (size_t)kv->layer * c->maxB * c->Hkv;
  const int ST = std::min(c->bs, c->sub_tile);
  RowArgs a{};
  if (int e = page_map(c, kv->k_pages, ST, &a.mapK)) return e;
  if (int e = page_map(c, kv->v_pages, ST, &a.mapV)) return e;
  a.table = kv->block_table; a.seq_lens = kv->seq_lens;
  a.app = (k_new && v_new) ? 1 : 0;
  a.k_new = (const uint16_t*)k_new; a.v_new = (const uint16_t*)v_new;
  a.kp_w = (uint16_t*)kv->k_pages; a.vp_w = (uint16_t*)kv->v_pages; a.summ_w = (uint4*)summaries;
  a.open_sum = c->open_sum + (size_t)kv->layer * c->maxB * c->Hkv * c->D; a.seq_lens_w = (int32_t*)kv->seq_lens;
  a.q = (const uint16_t*)q; a.summ = (const uint4*)summaries; a.out = out;
  a.done_host = c->arm_seq ? c->done_d : nullptr; a.done_seq = c->arm_seq; c->arm_seq = 0;
  a.scores = c->scores + r * c->MB;
  a.ema_l = c->ema_l + r * c->MB; a.ema_v = c->ema_v + r * c->MB;
  a.n_state = c->n_state + r;
  a.theta = c->theta + (size_t)kv->layer * c->maxB * 3;
  a.P0 = c->Pbuf[0] + r * c->Bud; a.P1 = c->Pbuf[1] + r * c->Bud; a.parity = c->parity + kv->layer;
  a.setA = c->setA + r * c->K; a.setM = c->setM + r * c->K; a.counts = c->counts + r * 3;
  a.ctl = c->ctl; a.stats = c->stats;
  a.tl = c->tl_on ? c->tl : nullptr;
  a.B = kv->batch; a.Hq = c->Hq; a.Hkv = c->Hkv; a.G = c->G; a.MB = c->MB; a.MBw = (c->MB + 31) / 32 + 1;
  a.bs = c->bs; a.K = c->K; a.Bud = c->Bud; a.NBH = c->MB; a.BudSel = c->bud_eff[kv->layer];
  a.BudMax = a.BudSel;
  for (int b = 0; b < kv->batch; ++b) {
    const int v = c->bud_seq_h[(size_t)kv->layer * c->maxB + b];
    if (v > 0) a.BudMax = std::max(a.BudMax, v - 1);
  }
  a.bud_seq = c->bud_seq + (size_t)kv->layer * c->maxB;
  a.retain = c->lay.overpredict_policy == PRR_RETAIN;
  a.spec = (spec && c->Bud > 0) ? 1 : 0;
  a.cut = c->cut;
  a.recompute = c->mode == PRR_MODE_S1 ? 1 : 0;
  a.scale = c->sm_scale; a.score_c = c->score_c;
  cudaError_t e = cudaErrorInvalidValue;
#define PRR_CASE(DD, SS) if (c->D == DD && ST == SS) e = plan_and_launch<DD, SS>(c, a, s);
  PRR_CASE(128, 64) PRR_CASE(128, 32) PRR_CASE(128, 16)
  PRR_CASE(64, 64) PRR_CASE(64, 32) PRR_CASE(64, 16)
#undef PRR_CASE
  c->launches++;
  return e == cudaSuccess ? 0 : (int)e;
}

}  // namespace prr
