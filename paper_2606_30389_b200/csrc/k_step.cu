// k_step — one PRR layer-step (a0-a8) as ONE persistent launch (Fig. 1, :38-42, :115 Fig. 5).
//
// The paper overlaps speculative attention with selection on two streams; on B200 a layer-step at
// batch 1 moves ~30 MB, i.e. ~5 us of HBM time, so kernel boundaries and launch gaps (2-3 us each)
// are the cost that matters.  Here the whole step is one grid of #SM CTAs whose WARPS are the
// workers: each warp owns a shared-memory tile buffer (K and V tile of one block, filled by TMA in
// the 128-byte swizzle) and walks through the phases below.  Dependencies between warps are
// epoch-valued flags in global memory (producer: stores, warp/CTA barrier, one st.release of the
// launch's epoch; consumer: ld.acquire polls of exactly the flags it needs, whole warps leaving on a
// vote).  Every wait targets an EARLIER phase of other warps and all CTAs are co-resident
// (cooperative launch), so the schedule cannot deadlock; waits are bounded anyway and raise
// ctl[CTL_ERR] (prr_check).  DESIGN.md section 8 has the measured timeline and what shaped it.
//
//   worker CTAs
//     phase 1  a0 + a1: one chunk of summary rows per warp, copied with cp.async into the warp's idle
//              tile buffer; exact fp64 accumulation (Q1); the warp whose chunk holds the open block
//              appends the new token (cache slot, fp64 running sum, summary row) and patches the
//              staged row; one flag per chunk.  No tile is requested before the SM has published.
//     phase 3  a4: the warp's speculative units, per-block partial state (m, l, O) of the blocks of P
//              (first wave paced at the HBM rate so the critical-path accesses are not queued behind it)
//     phase 4  a6: repair units, dealt out statically as (row, slot) tickets; the ticket's warp polls
//              its own epoch-tagged word of M and runs the same tile code
//     phase 5  a7: merge items (query head x 16-channel slice), dealt to the idle worker warps: wait
//              for the row's merge list, then for exactly the units in it (their tagged m words); fold hits u M (DROP) or
//              P u M (RETAIN) by Eq. 6-8, speculative entries first, one division at the end
//   job CTAs (one row job each when 2R <= #SM/4; otherwise the highest-numbered warps take the jobs)
//     phase 2  select(row): P as a bitmask, wait for the row's chunk flags, exact top-K on order-
//                           preserving keys in registers (a2), M = A\P (a5) published first, then
//                           the merge list, then A / bitmask / counters
//              ema(row):    (l, v) staged in shared memory meanwhile; Eq. 3 update, Eq. 2 prediction,
//                           top-Bud -> P of the NEXT step into the other parity buffer (a8, a3)
//   exit       the last warp bumps the epoch, flips the layer's P parity and (fused append) seq_lens
//
// spec = 0 runs the same kernel as the sequential select-then-attend path: P is
// treated as empty, every block of A is a "repair" unit that can only start after selection.
#include <cuda.h>
#include <math_constants.h>

#include <cstdlib>
#include <cstring>

#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {
namespace persist {  // (k_row.cu has its own tile / selection code: keep the two apart)

constexpr float LOG2E_F = 1.4426950408889634f;
constexpr uint32_t SPIN_LIMIT = 1u << 22;  // ~0.1-0.5 s of polling, then give up loudly

// Dependencies between warps are epoch-valued FLAGS, not counters: a producer publishes with one
// st.release of the launch's epoch (no atomics, nothing to reset), a consumer polls exactly the
// flags of the items it needs.  ctl = header, then sel[Rmax] (A, M, counters written), sel2[Rmax] x 64 bit (epoch << 32 | list lengths: merge
// list written), spec-unit flags [Rmax*Bud], repair-unit flags [Rmax*K], score-chunk flags [Rmax*MB].
enum { CTL_EXIT = 0, CTL_ERR = 1, CTL_EPOCH = 2, CTL_HDR = 8 };

__device__ __forceinline__ uint32_t ld_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned long long gtime() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;\n" : "=l"(t));
  return t;
}

__device__ __forceinline__ unsigned long long ld_relaxed64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];\n" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_relaxed64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;\n" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void st_release64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;\n" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];\n" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}
// One thread spins until *p == v (acquire).  Bounded: gives up loudly.
__device__ __forceinline__ void spin_eq(const uint32_t* p, uint32_t v, uint32_t* err) {
  uint32_t it = 0;
  while (ld_acquire(p) != v) {
    __nanosleep(20);
    if (++it > SPIN_LIMIT) { atomicExch(err, 1u); break; }
  }
}
// Warp-collective wait until *p == v.  Lane 0 polls; __syncwarp orders the other lanes after it.
__device__ __forceinline__ void wait_eq(const uint32_t* p, uint32_t v, uint32_t* err) {
  if ((threadIdx.x & 31) == 0) spin_eq(p, v, err);
  __syncwarp();
}
// Warp-collective wait until f[0 .. n) all equal v.  The warp stays converged: every lane polls up
// to four flags per round trip and the loop exits on a vote (lanes spinning in private loops would
// be serialised).
__device__ __forceinline__ void wait_flags(const uint32_t* f, int n, uint32_t v, uint32_t* err) {
  const int lane = threadIdx.x & 31;
#pragma unroll 1
  for (int base = 0; base < n; base += 128) {
    uint32_t it = 0;
#pragma unroll 1
    for (;;) {
      bool ok = true;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int c = base + lane + 32 * k;
        if (c < n) ok = ok && (ld_acquire(f + c) == v);
      }
      if (__all_sync(FULL, ok)) break;
      __nanosleep(20);
      if (++it > SPIN_LIMIT) { if (lane == 0) atomicExch(err, 1u); break; }
    }
  }
}
// Warp-collective publish: the lanes' earlier stores are ordered before lane 0's release by the
// warp barrier (the release is cumulative over it).
__device__ __forceinline__ void signal_set(uint32_t* p, uint32_t v) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) st_release(p, v);
}

struct Thr { uint32_t key; int idx; };  // selected(i) <=> key_i > key || (key_i == key && i <= idx)
__device__ __forceinline__ bool selected(uint32_t key, int i, const Thr& t) {
  return key > t.key || (key == t.key && i <= t.idx);
}

// ---------------------------------------------------------------------------------------------
// A team is the set of threads that works on one row job: a whole CTA or one warp.
struct Team {
  int tid, nt, wid, nw;
  bool cta;
  __device__ __forceinline__ void sync() const { if (cta) __syncthreads(); else __syncwarp(); }
};
// The team's shared memory: the row's keys (if they fit), bitmask / offset words, a histogram of
// 2^hbits counters, reduction slots.
struct TeamMem {
  uint32_t* keys; int key_cap;
  uint32_t *pmask, *amask, *offs;  // [MBw] each
  uint32_t* hist; int hbits;       // [1 << hbits], zero on entry to and exit from team_kth
  uint32_t* red;                   // [nw*16] per-warp slots, then 8 decision words
  unsigned long long* cand;        // [CAND] candidates (key << 32 | ~index), 8-byte aligned
  uint32_t* rk;                    // [CAND] partial ranks, zero between uses
  int32_t* plist;                  // [Bud] the predicted blocks by slot (select jobs)
  double *Ls, *Vs; int st_cap;     // staged EMA state of the row [st_cap] each (8-byte aligned)
};
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void red_shared_add(uint32_t* p, uint32_t v) {
  asm volatile("red.shared.add.u32 [%0], %1;\n" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
struct Keys {  // the row's order-preserving keys: shared memory if they fit, else recomputed from global
  uint32_t sm; const float* gl;  // sm: shared-window address of keys[0], 0 = not resident
  __device__ __forceinline__ uint32_t get(int i) const {
    return sm ? lds_u32(sm + 4u * (uint32_t)i) : score_key(__ldcg(gl + i));
  }
};

// Highest bucket b of hist[0 .. NB) with  sum_{b' >= b} hist[b'] >= need  (1 <= need <= total);
// `above` = the count in the buckets over b.  Thread t owns the buckets [NB-(t+1)per, NB-t*per), so
// a prefix scan over threads is a suffix scan over buckets.  Every thread zeroes the buckets it
// read; every thread returns the same triple.
__device__ void team_pick(uint32_t* hist, int NB, int need, const Team& tm, const TeamMem& m, int& bstar,
                          int& cstar, int& above) {
  const int lane = threadIdx.x & 31;
  uint32_t* dec = m.red + tm.nw * 16;
  const int per = (NB + tm.nt - 1) / tm.nt;
  const int hi = NB - tm.tid * per, lo = max(0, hi - per);
  uint32_t sum = 0;
#pragma unroll 4
  for (int b = lo; b < hi; ++b) sum += hist[b];
  uint32_t incl = sum;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const uint32_t x = __shfl_up_sync(FULL, incl, off);
    if (lane >= off) incl += x;
  }
  if (tm.cta) {
    if (lane == 31) m.red[tm.wid] = incl;
    __syncthreads();
#pragma unroll 1
    for (int w = 0; w < tm.wid; ++w) incl += m.red[w];
  }
  const uint32_t excl = incl - sum;
  if ((int)excl < need && need <= (int)incl) {  // the crossing is in this thread's buckets (exactly one thread)
    uint32_t acc = excl;
#pragma unroll 1
    for (int b = hi - 1; b >= lo; --b) {
      const uint32_t c = hist[b];
      if ((int)(acc + c) >= need) { dec[0] = (uint32_t)b; dec[1] = c; dec[2] = acc; break; }
      acc += c;
    }
  }
#pragma unroll 1
  for (int b = lo; b < hi; ++b) hist[b] = 0u;
  tm.sync();
  bstar = (int)dec[0]; cstar = (int)dec[1]; above = (int)dec[2];
}

// ---------------------------------------------------------------------------------------------
// Exact k-th largest of n keys under the order (key desc, index asc), by one team, as a threshold
// pair.  Range narrowing on the order-preserving keys: the invariant is "the threshold key lies in
// [lo, lo+span]; `need` of the keys in that range are selected, every key above it is".  Each pass
// histograms the range into 2^hbits buckets (shared-memory reductions) and keeps the bucket the
// threshold falls in; <= 64 survivors are ranked directly; a range of one key value is resolved by
// index order.  Integer-only, hence order-independent and bit-exact (Q4).  Requires
// 1 <= k < n, [lo, lo+span] = the exact key range of the row, and a zeroed histogram.
// ---------------------------------------------------------------------------------------------
constexpr int CAND = 128;  // survivors that are ranked directly
constexpr uint32_t MERGE_END = 0x7fffffffu;  // tagged merge list: no entry here

// The need-th (1-based) of the cnt candidates under (key desc, index asc).  A candidate is one
// 64-bit word (key << 32 | ~index): larger word = better.  All threads work: the comparisons of a
// candidate are split over nt / cnt threads whose partial ranks meet in shared memory (rk[], zero on
// entry and on exit).
__device__ __forceinline__ Thr team_rank(int cnt, int need, const Team& tm, const TeamMem& m) {
  uint32_t* dec = m.red + tm.nw * 16;
  if (tm.nt >= cnt) {  // (uniform) a candidate's comparisons are split over nt / cnt threads
    const int parts = tm.nt / cnt;
    const int e = tm.tid % cnt, p = tm.tid / cnt;
    unsigned long long ce = 0ull;
    if (p < parts) {
      ce = m.cand[e];
      const int per = (cnt + parts - 1) / parts;
      const int f0 = p * per, f1 = min(cnt, f0 + per);
      uint32_t rank = 0;
#pragma unroll 4
      for (int f = f0; f < f1; ++f) rank += m.cand[f] > ce;
      if (parts > 1) atomicAdd(&m.rk[e], rank); else m.rk[e] = rank;
    }
    tm.sync();
    if (p == 0) {
      if ((int)m.rk[e] == need - 1) { dec[5] = (uint32_t)(ce >> 32); dec[6] = ~(uint32_t)ce; }  // exactly one
      m.rk[e] = 0u;
    }
  } else {             // fewer threads than candidates: a thread ranks several
#pragma unroll 1
    for (int e = tm.tid; e < cnt; e += tm.nt) {
      const unsigned long long ce = m.cand[e];
      uint32_t rank = 0;
#pragma unroll 4
      for (int f = 0; f < cnt; ++f) rank += m.cand[f] > ce;
      if ((int)rank == need - 1) { dec[5] = (uint32_t)(ce >> 32); dec[6] = ~(uint32_t)ce; }
    }
  }
  tm.sync();
  Thr r;
  r.key = dec[5]; r.idx = (int)dec[6];
  tm.sync();
  return r;
}

__device__ Thr team_kth(const Keys& ks, int n, int k, const Team& tm, const TeamMem& m, uint32_t lo, uint32_t span,
                        int cnt_in) {
  const int lane = threadIdx.x & 31;
  uint32_t* dec = m.red + tm.nw * 16;  // [0] bstar [1] cstar [2] acc [5] key [6] idx [7] cand count
  int need = k;
  Thr r;
  for (;;) {
    if (span == 0) {  // all survivors share one key: the `need` lowest indices win
      if (tm.wid == 0) {
        int base = 0, idx = n - 1;
#pragma unroll 1
        for (int j0 = 0; j0 < n; j0 += 32) {
          const int i = j0 + lane;
          const uint32_t bal = __ballot_sync(FULL, i < n && ks.get(i) == lo);
          const int c = __popc(bal);
          if (base + c >= need) { idx = j0 + (int)__fns(bal, 0, need - base); break; }
          base += c;
        }
        if (lane == 0) { dec[5] = lo; dec[6] = (uint32_t)idx; }
      }
      tm.sync();
      r.key = dec[5]; r.idx = (int)dec[6];
      tm.sync();
      return r;
    }
    if (cnt_in <= CAND) {  // collect the survivors (any order) and rank them
      if (tm.tid == 0) dec[7] = 0u;
      tm.sync();
#pragma unroll 4
      for (int i = tm.tid; i < n; i += tm.nt) {
        const uint32_t key = ks.get(i);
        if ((key - lo) <= span) {
          const uint32_t pos = atomicAdd(&dec[7], 1u);
          m.cand[pos] = ((unsigned long long)key << 32) | (uint32_t)~i;
        }
      }
      tm.sync();
      return team_rank(cnt_in, need, tm, m);
    }
    const int sh = max(0, (32 - __clz(span)) - m.hbits);  // (span >> sh) < 2^hbits
#pragma unroll 4
    for (int i = tm.tid; i < n; i += tm.nt) {
      const uint32_t d = ks.get(i) - lo;
      if (d <= span) red_shared_add(&m.hist[d >> sh], 1u);
    }
    tm.sync();
    int bstar, cstar, acc;
    team_pick(m.hist, 1 << m.hbits, need, tm, m, bstar, cstar, acc);
    need -= acc;
    cnt_in = cstar;
    const uint32_t off = (uint32_t)bstar << sh;
    const uint32_t width = sh ? ((1u << sh) - 1u) : 0u;
    lo += off;
    span = min(span - off, width);
    if (need == cnt_in) { r.key = lo; r.idx = 0x7fffffff; return r; }  // the whole sub-range is selected
  }
}

// Team-wide min / max of the per-thread key range -> (lo, span).
__device__ __forceinline__ void team_range(uint32_t kmin, uint32_t kmax, const Team& tm, const TeamMem& m,
                                           uint32_t& lo, uint32_t& span) {
  kmin = __reduce_min_sync(FULL, kmin);
  kmax = __reduce_max_sync(FULL, kmax);
  if (!tm.cta) { lo = kmin; span = kmax >= kmin ? kmax - kmin : 0u; return; }
  if ((threadIdx.x & 31) == 0) { m.red[tm.wid * 2] = kmin; m.red[tm.wid * 2 + 1] = kmax; }
  tm.sync();
#pragma unroll 1
  for (int w = 0; w < tm.nw; ++w) { kmin = min(kmin, m.red[w * 2]); kmax = max(kmax, m.red[w * 2 + 1]); }
  tm.sync();
  lo = kmin; span = kmax >= kmin ? kmax - kmin : 0u;
}

// Ordered emission: the selected indices ascending into list[width] (padded with -1), the bitmask
// into mask_g (global, may be null); with Mlist != null also the selected indices NOT in pmask
// (ascending, padded to widthM).  Returns (nA << 16) | nM in every thread.
__device__ uint32_t team_emit(const Keys& ks, int n, int k, const Thr& t, const Team& tm, const TeamMem& m,
                              int32_t* list, int width, uint32_t* mask_g, int32_t* Mlist, int widthM) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  const int nwd = (n + 31) >> 5;
  uint32_t* dec = m.red + tm.nw * 16;
#pragma unroll 4
  for (int w = tm.wid; w < nwd; w += tm.nw) {
    const int i = w * 32 + lane;
    const bool sel = i < n && k > 0 && selected(ks.get(i), i, t);
    const uint32_t aw = __ballot_sync(FULL, sel);
    if (lane == 0) m.amask[w] = aw;
  }
  tm.sync();
  if (tm.wid == 0) {
    uint32_t carry = 0;
#pragma unroll 1
    for (int w0 = 0; w0 < nwd; w0 += 32) {
      const int w = w0 + lane;
      const uint32_t aw = w < nwd ? m.amask[w] : 0u;
      const uint32_t mw = (Mlist && w < nwd) ? (aw & ~m.pmask[w]) : 0u;
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
  tm.sync();
#pragma unroll 2
  for (int w = tm.wid; w < nwd; w += tm.nw) {
    const uint32_t aw = m.amask[w];
    const uint32_t off = m.offs[w];
    const int i = w * 32 + lane;
    if ((aw >> lane) & 1u) {
      list[(off >> 16) + __popc(aw & lt)] = i;
      if (Mlist) {
        const uint32_t mw = aw & ~m.pmask[w];
        if ((mw >> lane) & 1u) Mlist[(off & 0xffffu) + __popc(mw & lt)] = i;
      }
    }
    if (mask_g && lane == 0) mask_g[w] = aw;
  }
  const uint32_t tot = dec[3];
#pragma unroll 1
  for (int j = (int)(tot >> 16) + tm.tid; j < width; j += tm.nt) list[j] = -1;
  if (Mlist)
#pragma unroll 1
    for (int j = (int)(tot & 0xffffu) + tm.tid; j < widthM; j += tm.nt) Mlist[j] = -1;
  tm.sync();
  return tot;
}

// ---------------------------------------------------------------------------------------------
struct StepArgs;
__device__ __forceinline__ int seq_len(const StepArgs& a, int b);
struct StepArgs {
  alignas(64) CUtensorMap mapK;  // bf16 [rows = n_pages*Hkv*bs, d], box [bs, 64], 128-byte swizzle
  alignas(64) CUtensorMap mapV;
  const uint16_t* kp; const uint16_t* vp; const int32_t* table; const int32_t* seq_lens;
  // fused append (a0): app = 1 -> seq_lens holds the lengths BEFORE the append, every length below is +1
  const uint16_t* k_new; const uint16_t* v_new; uint16_t* kp_w; uint16_t* vp_w; uint4* summ_w; double* open_sum;
  int32_t* seq_lens_w; int app;
  const uint16_t* q; const uint4* summ; float* out;
  // layer state (already offset to the layer)
  float* scores; double* ema_l; double* ema_v; int32_t* n_state; const double* theta;
  int32_t* P0; int32_t* P1; int32_t* parity;
  int32_t* setA; int32_t* setM; int32_t* counts;
  // per-step scratch
  uint32_t* maskA; float* pred; uint32_t* msrc; int32_t* mn;
  // M as self-describing words, one per (row, repair slot): epoch << 32 | block + 1 (0 = no such miss).  A
  // repair warp polls ITS word: no flag, no fence and no second load between selection and the tile request.
  unsigned long long* mtag;
  // the step's scores once more as self-describing words (epoch << 32 | fp32 bits), [Rmax, MB]: a row job in
  // the fast path polls its own words instead of chunk flags: no producer fence and no flag -> data round trip
  unsigned long long* sc64;
  // the merge lists once more as self-describing words (epoch << 32 | slot code, MERGE_END past the end),
  // [Rmax, Bud + K]: a merge warp polls the list itself -- no flag, no producer fence, no second load
  unsigned long long* ms64;
  float* O_spec; float* m_spec; float* l_spec; float* O_rep; float* m_rep; float* l_rep;
  // a unit's block-local maxima as self-describing words (epoch << 32 | fp32 bits of m), one per (query head,
  // slot), written with st.release after the unit's partial rows and l: the word is the unit's "done" flag AND m
  unsigned long long* mt_spec; unsigned long long* mt_rep;
  uint32_t* ctl; uint32_t* sel; unsigned long long* sel2; uint32_t* ufs; uint32_t* ufr; uint32_t* sfl;  // header, then the flag arrays
  unsigned long long* stats; unsigned long long* tl;
  int B, Hq, Hkv, G, MB, MBw, bs, K, Bud, BudSel, Rmax, retain, spec, buf_bytes, scr_bytes, J, CR;  // BudSel <= Bud: the run-time budget of the NEXT prediction
  int msw;  // channels per merge item (16 .. D): the narrowest slice that still gives every merge warp at most one item
  float scale; float pace_ns; double score_c;
  uint32_t* done_host; uint32_t done_seq;  // host-visible completion word (mapped host memory) and its value, or null
  const int32_t* bud_seq;  // per sequence of the layer: 0 = the layer's budget, v > 0 = budget v - 1 (prr_set_budget_seq)
};

__device__ __forceinline__ int seq_len(const StepArgs& a, int b) { return __ldcg(a.seq_lens + b) + a.app; }

template <int D, int BS>
struct Tile {
  // Shared-memory image of one (block, KV head) tile as the copy engine writes it: the K half then
  // the V half, each D/64 boxes of [BS rows x 128 bytes] in the 128-byte swizzle (the 16-byte
  // chunk c of row r sits at chunk c ^ (r & 7)), so ldmatrix is conflict-free without padding.
  static constexpr int NBOX = D / 64;
  static constexpr int BOX_BYTES = BS * 128;
  static constexpr int HALF = NBOX * BOX_BYTES;  // = BS * D * 2
  static constexpr int BYTES = 2 * HALF;         // K tile + V tile
  static constexpr int SUB = BS < 64 ? BS : 64;  // tokens per softmax sub-tile
  static constexpr int WFIT = (216 * 1024) / (BYTES + 1024);
  static constexpr int WMAX = WFIT < 12 ? WFIT : 12;  // warps per CTA (one tile buffer each)
  __device__ static __forceinline__ const unsigned char* at(const unsigned char* half, int r, int c) {
    return half + (c >> 3) * BOX_BYTES + r * 128 + (((c & 7) ^ (r & 7)) << 4);
  }
};

// Put the TMA loads of one (block, KV head) tile in flight: bars[0] completes when K has landed,
// bars[1] when V has, so QK^T can start while V is still in flight.  The whole block is fetched;
// rows >= valid (unwritten cache slots of the open block) are masked / zeroed by tile_compute.
template <int D, int BS>
__device__ __forceinline__ void tile_load(unsigned char* Ks, unsigned long long* bars, const StepArgs& a, int page,
                                          int h) {
  using T = Tile<D, BS>;
  fence_proxy_async();  // this buffer was last touched through the generic proxy
  __syncwarp();
  if ((threadIdx.x & 31) == 0) {
    const int y = (page * a.Hkv + h) * BS;
    mbar_expect_tx(&bars[0], T::HALF);
#pragma unroll
    for (int i = 0; i < T::NBOX; ++i) tma_load_2d(Ks + i * T::BOX_BYTES, &a.mapK, i * 64, y, &bars[0]);
    mbar_expect_tx(&bars[1], T::HALF);
#pragma unroll
    for (int i = 0; i < T::NBOX; ++i) tma_load_2d(Ks + T::HALF + i * T::BOX_BYTES, &a.mapV, i * 64, y, &bars[1]);
  }
}

// Per-block partial state (the forward also writes l and m) by ONE warp from its
// landed tile: S = Q K^T on mma.sync m16n8k16 (the G <= 16 query heads of the group are the M rows,
// zero padded), block-local max / sum with quad shuffles, P V with P as a two-term bf16 split.
// The state is relative to the BLOCK-LOCAL maximum, so a block's partial is the same bits whether
// it was computed speculatively, as a repair, or by the sequential path.
template <int D, int BS>
__device__ __forceinline__ void tile_compute(unsigned char* Ks, unsigned long long* bars, uint32_t phase,
                                             const StepArgs& a, int b, int h, int valid, float* O, unsigned long long* Mt,
                                             float* Lo, int width, int slot, const uint16_t* patch_k,
                                             const uint16_t* patch_v, uint32_t ep) {
  using T = Tile<D, BS>;
  constexpr int SUB = T::SUB, NT8 = SUB / 8;
  unsigned char* Vs = Ks + T::HALF;
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

  mbar_wait(&bars[0], phase);  // K landed
  if (patch_k) {  // fused append: the token appended by this launch is not in the cache yet
    if (lane < D / 8)
      *reinterpret_cast<uint4*>(const_cast<unsigned char*>(T::at(Ks, valid - 1, lane))) =
          __ldg(reinterpret_cast<const uint4*>(patch_k) + lane);
    __syncwarp();
  }
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
        ldmatrix_x4(b0, b1, b2, b3, T::at(Ks, tok0 + nt * 8 + rr, k2 * 4 + mat));
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
    if (st == 0) {
      mbar_wait(&bars[1], phase);  // V landed
      if (patch_v) {
        if (lane < D / 8)
          *reinterpret_cast<uint4*>(const_cast<unsigned char*>(T::at(Vs, valid - 1, lane))) =
              __ldg(reinterpret_cast<const uint4*>(patch_v) + lane);
        __syncwarp();
      }
      if (valid < BS) {            // open block: 0 * (whatever an unwritten slot holds) must not reach P V
        for (int i = lane; i < (BS - valid) * T::NBOX * 8; i += 32) {
          const int r = valid + i / (T::NBOX * 8), c = i % (T::NBOX * 8);
          *reinterpret_cast<uint4*>(Vs + (c >> 3) * T::BOX_BYTES + r * 128 + ((c & 7) << 4)) = make_uint4(0, 0, 0, 0);
        }
        __syncwarp();
      }
    }
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
                          T::at(Vs, tok0 + kk * 16 + (mat & 1) * 8 + rr, d2 * 2 + (mat >> 1)));
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
    if (tq == 0) Lo[st] = l0;
  }
  if (r0 + 8 < G) {
    const size_t st = (hb + r0 + 8) * width + slot;
#pragma unroll
    for (int dt = 0; dt < D / 8; ++dt)
      *reinterpret_cast<float2*>(O + st * D + dt * 8 + tq * 2) = make_float2(o[dt][2], o[dt][3]);
    if (tq == 0) Lo[st] = l1;
  }
  // publish: every lane's partial rows and l are ordered before the releases by the warp barrier (the
  // release is cumulative over it); the tagged m IS the unit's completion flag for that query head
  __syncwarp();
  const unsigned long long tag = (unsigned long long)ep << 32;
  if (tq == 0 && r0 < G) st_release64(Mt + (hb + r0) * width + slot, tag | __float_as_uint(mrun0 * a.scale));
  if (tq == 0 && r0 + 8 < G) st_release64(Mt + (hb + r0 + 8) * width + slot, tag | __float_as_uint(mrun1 * a.scale));
}

// ---------------------------------------------------------------------------------------------
// a1: summary rows [r0, end) of (b, h) by one warp.  The rows are copied to the warp's own (still
// idle) tile buffer with cp.async -- every 16-byte request of the chunk is in flight at once and
// the code stays a short rolled loop (instruction cache) -- then sub-warps of D/8 lanes take a row
// each: the group's queries are pre-summed per channel in fp64, products and sums are exact (Q1).
template <int D>
__device__ __forceinline__ int score_chunk(const StepArgs& a, int b, int h, int r0, int end_ld, unsigned char* stage,
                                           uint32_t ep, unsigned long long* tl) {
  constexpr int LPR = D / 8, RW = 32 / LPR;
  const int lane = threadIdx.x & 31, sub = lane / LPR, l = lane % LPR;
  const uint4* rows = a.summ + (((size_t)b * a.Hkv + h) * a.MB + r0) * LPR + l;
  float* out = a.scores + ((size_t)b * a.Hkv + h) * a.MB + r0;
  unsigned long long* out64 = a.sc64 + ((size_t)b * a.Hkv + h) * a.MB + r0;
  // The copies do not wait for the sequence length: rows up to the chunk's end inside the summary
  // buffer are fetched (rows past the last block hold stale data and are never scored).
  const int nld = end_ld - r0;
  uint4* st = reinterpret_cast<uint4*>(stage) + l;
#pragma unroll 4
  for (int r = sub; r < nld; r += RW) cp_async16(st + r * LPR, rows + (size_t)r * LPR);
  cp_async_commit();
  if (tl && lane == 0) tl[12] = gtime();
  const int len = seq_len(a, b);
  // the group's queries summed per channel (exact in fp64): the 8 channels this lane owns
  double qs[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) qs[j] = 0.0;
  const uint16_t* qb = a.q + ((size_t)b * a.Hq + (size_t)h * a.G) * D + l * 8;
#pragma unroll 1
  for (int g0 = 0; g0 < a.G; g0 += 4) {  // four query rows per batch of loads (zeros add nothing)
    uint4 t[4];
#pragma unroll
    for (int e = 0; e < 4; ++e)
      t[e] = g0 + e < a.G ? __ldg(reinterpret_cast<const uint4*>(qb + (size_t)(g0 + e) * D)) : make_uint4(0, 0, 0, 0);
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
  const int nb = max(0, min(a.MB, (len + a.bs - 1) / a.bs));
  const int nr = min(end_ld, nb) - r0;
  if (tl && lane == 0) tl[6] = gtime();
  cp_async_wait<0>();
  __syncwarp();
  if (tl && lane == 0) tl[13] = gtime();
  if (a.app) {
    // a0: the warp that scores the block the new token falls in appends it: cache slot, running sum
    // and mean-key summary (exact fp64 sum, one division, one RNE to bf16, Q2) -- and patches the
    // summary row it has just staged, so the score below is the score after the append.
    const int pos = len - 1, ob = pos / a.bs, slot = pos - ob * a.bs;
    if (ob >= r0 && ob < r0 + nr && sub == 0) {
      const size_t ch = ((size_t)b * a.Hkv + h) * D + l * 8;
      const uint4 kn = __ldg(reinterpret_cast<const uint4*>(a.k_new + ch));
      const uint4 vn = __ldg(reinterpret_cast<const uint4*>(a.v_new + ch));
      const size_t page = (size_t)__ldg(a.table + (size_t)b * a.MB + ob);
      const size_t dst = ((page * a.Hkv + h) * a.bs + slot) * (size_t)D + l * 8;
      *reinterpret_cast<uint4*>(a.kp_w + dst) = kn;
      *reinterpret_cast<uint4*>(a.vp_w + dst) = vn;
      const uint32_t w[4] = {kn.x, kn.y, kn.z, kn.w};
      uint32_t o[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const double x0 = (double)bf16_lo(w[j]), x1 = (double)bf16_hi(w[j]);
        const double s0 = slot == 0 ? x0 : __dadd_rn(a.open_sum[ch + 2 * j], x0);
        const double s1 = slot == 0 ? x1 : __dadd_rn(a.open_sum[ch + 2 * j + 1], x1);
        a.open_sum[ch + 2 * j] = s0;
        a.open_sum[ch + 2 * j + 1] = s1;
        o[j] = (uint32_t)f64_to_bf16_rne(__ddiv_rn(s0, (double)(slot + 1))) |
               ((uint32_t)f64_to_bf16_rne(__ddiv_rn(s1, (double)(slot + 1))) << 16);
      }
      const uint4 row = make_uint4(o[0], o[1], o[2], o[3]);
      st[(ob - r0) * LPR] = row;
      a.summ_w[(((size_t)b * a.Hkv + h) * a.MB + ob) * LPR + l] = row;
    }
    __syncwarp();
  }
  // Eight rows per trip and per sub-warp (four in a short last trip).  The per-lane partial sums are
  // folded across the LPR lanes by a transposed butterfly (each step halves what a lane carries): 7-8
  // 64-bit shuffles instead of 8 x log2(LPR).  Every partial sum is exact (Q1), so the order of
  // accumulation is free.
  auto dot = [&](int r) -> double {
    const uint4 v = r < nr ? st[r * LPR] : make_uint4(0, 0, 0, 0);
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    double a0 = 0.0, a1 = 0.0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      a0 = fma((double)bf16_lo(w[j]), qs[2 * j], a0);
      a1 = fma((double)bf16_hi(w[j]), qs[2 * j + 1], a1);
    }
    return a0 + a1;
  };
  const bool upA = (l & (LPR / 2)) != 0, upB = (l & (LPR / 4)) != 0, upC = (l & (LPR / 8)) != 0;
  int rr0 = 0;
#pragma unroll 1
  for (; nr - rr0 > 4 * RW; rr0 += 8 * RW) {  // warp-uniform trip counts (full-mask shuffles below)
    double acc[8], v4[4], v2[2];
#pragma unroll
    for (int e = 0; e < 8; ++e) acc[e] = dot(rr0 + e * RW + sub);
#pragma unroll
    for (int j = 0; j < 4; ++j)
      v4[j] = (upA ? acc[4 + j] : acc[j]) + __shfl_xor_sync(FULL, upA ? acc[j] : acc[4 + j], LPR / 2);
#pragma unroll
    for (int j = 0; j < 2; ++j)
      v2[j] = (upB ? v4[2 + j] : v4[j]) + __shfl_xor_sync(FULL, upB ? v4[j] : v4[2 + j], LPR / 4);
    double v1 = (upC ? v2[1] : v2[0]) + __shfl_xor_sync(FULL, upC ? v2[0] : v2[1], LPR / 8);
    if (LPR == 16) v1 += __shfl_xor_sync(FULL, v1, 1);
    const int r = rr0 + ((upA ? 4 : 0) + (upB ? 2 : 0) + (upC ? 1 : 0)) * RW + sub;
    if (r < nr && (LPR == 8 || (l & 1) == 0)) {
      const float sv = f64_to_score(__dmul_rn(v1, a.score_c));
      st_relaxed64(out64 + r, ((unsigned long long)ep << 32) | __float_as_uint(sv));
      out[r] = sv;
    }
  }
  if (rr0 < nr) {  // at most 4 * RW rows left
    double acc[4], v2[2];
#pragma unroll
    for (int e = 0; e < 4; ++e) acc[e] = dot(rr0 + e * RW + sub);
#pragma unroll
    for (int j = 0; j < 2; ++j)
      v2[j] = (upA ? acc[2 + j] : acc[j]) + __shfl_xor_sync(FULL, upA ? acc[j] : acc[2 + j], LPR / 2);
    double v1 = (upB ? v2[1] : v2[0]) + __shfl_xor_sync(FULL, upB ? v2[0] : v2[1], LPR / 4);
#pragma unroll
    for (int off = LPR / 8; off >= 1; off >>= 1) v1 += __shfl_xor_sync(FULL, v1, off);
    const int r = rr0 + ((upA ? 2 : 0) + (upB ? 1 : 0)) * RW + sub;
    if (r < nr && (l & (LPR / 4 - 1)) == 0) {
      const float sv = f64_to_score(__dmul_rn(v1, a.score_c));
      st_relaxed64(out64 + r, ((unsigned long long)ep << 32) | __float_as_uint(sv));
      out[r] = sv;
    }
  }
  __syncwarp();
  return nb;
}

// ---------------------------------------------------------------------------------------------
// Fast path of the selection for rows with n <= KB * team threads (every config of BASELINE.json):
// thread t holds the keys of the blocks t, t + nt, ... in REGISTERS, so the passes below are
// straight-line predicated code without shared-memory round trips or per-element branches.  The
// results are the same exact (key desc, index asc) selection; rows that do not fit, or whose first
// pass leaves more than CAND candidates, continue in the generic code (team_kth / team_emit).
constexpr int KB = 12;

// First pass with a fixed bucket map (the top hbits of the key: monotone in the key), then the
// survivors are ranked directly.  k < n.
__device__ __forceinline__ Thr fast_kth(const uint32_t (&key)[KB], const Keys& ks, int n, int k, const Team& tm,
                                        const TeamMem& m, unsigned long long* tl) {
  uint32_t* dec = m.red + tm.nw * 16;
  const int sh = 32 - m.hbits;
#pragma unroll
  for (int e = 0; e < KB; ++e) {
    const int i = tm.tid + e * tm.nt;
    if (i < n) red_shared_add(&m.hist[key[e] >> sh], 1u);
  }
  if (tm.tid == 0) dec[7] = 0u;
  tm.sync();
  if (tl && tm.tid == 0) tl[12] = gtime();
  int bstar, cstar, acc;
  team_pick(m.hist, 1 << m.hbits, k, tm, m, bstar, cstar, acc);
  if (tl && tm.tid == 0) tl[13] = gtime();
  const int need = k - acc;
  const uint32_t lo = (uint32_t)bstar << sh, span = (1u << sh) - 1u;
  Thr r;
  if (need == cstar) { r.key = lo; r.idx = 0x7fffffff; return r; }  // the whole bucket is selected
  if (cstar > CAND) return team_kth(ks, n, need, tm, m, lo, span, cstar);
#pragma unroll
  for (int e = 0; e < KB; ++e) {
    const int i = tm.tid + e * tm.nt;
    if (i < n && (key[e] - lo) <= span) {
      const uint32_t pos = atomicAdd(&dec[7], 1u);
      m.cand[pos] = ((unsigned long long)key[e] << 32) | (uint32_t)~i;
    }
  }
  tm.sync();
  if (tl && tm.tid == 0) tl[14] = gtime();
  return team_rank(cstar, need, tm, m);
}

// The row's merge list (warp 0 of the team): hit slots (all of P when retained) ascending, then the
// repair slots; needs the bitmask of A in m.amask and the predicted blocks by slot in m.plist.
__device__ __forceinline__ uint32_t write_merge_list(const StepArgs& a, int row, int nb, int nM, const TeamMem& m,
                                                     uint32_t ep) {
  const int lane = threadIdx.x & 31;
  uint32_t* ms = a.msrc + (size_t)row * (a.Bud + a.K);
  unsigned long long* m64 = a.ms64 + (size_t)row * (a.Bud + a.K);
  const unsigned long long tag = (unsigned long long)ep << 32;
  int base = 0;
  if (a.spec) {
    for (int j0 = 0; j0 < a.Bud; j0 += 32) {
      const int j = j0 + lane;
      const int blk = j < a.Bud ? m.plist[j] : -1;
      const bool use = blk >= 0 && (a.retain || ((blk >> 5) < ((nb + 31) >> 5) && ((m.amask[blk >> 5] >> (blk & 31)) & 1u)));
      const uint32_t bal = __ballot_sync(FULL, use);
      if (use) {
        const int pos = base + __popc(bal & ((1u << lane) - 1u));
        ms[pos] = (uint32_t)j;
        st_relaxed64(m64 + pos, tag | (uint32_t)j);
      }
      base += __popc(bal);
    }
  }
  for (int j = lane; j < nM; j += 32) {
    ms[base + j] = (uint32_t)j | 0x80000000u;
    st_relaxed64(m64 + base + j, tag | (uint32_t)j | 0x80000000u);
  }
  for (int j = base + nM + lane; j < a.Bud + a.K; j += 32) st_relaxed64(m64 + j, tag | MERGE_END);
  const uint32_t pk = ((uint32_t)base << 16) | (uint32_t)(base + nM);  // speculative entries | all entries
  if (lane == 0) a.mn[row] = (int32_t)pk;
  return pk;  // travels with the flag (sel2), so the merge needs no load for it
}

// Ordered emission from the registers (see team_emit for the outputs).
__device__ __forceinline__ uint32_t fast_emit(const uint32_t (&key)[KB], int n, int k, const Thr& t, const Team& tm,
                                              const TeamMem& m, int32_t* list, int width, uint32_t* mask_g,
                                              int32_t* Mlist, int widthM, unsigned long long* mtag, uint32_t ep,
                                              const StepArgs& a, int row, int nb, unsigned long long* tl) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  const int nwd = (n + 31) >> 5, nw32 = tm.nt >> 5;
  uint32_t* dec = m.red + tm.nw * 16;
  uint32_t bal[KB], mwd[KB];
#pragma unroll
  for (int e = 0; e < KB; ++e) {  // lanes of a warp hold 32 consecutive blocks: one mask word per (warp, e)
    const int i = tm.tid + e * tm.nt, w = tm.wid + e * nw32;
    const bool sel = i < n && k > 0 && selected(key[e], i, t);
    bal[e] = __ballot_sync(FULL, sel);
    mwd[e] = 0u;
    if (w < nwd) {
      if (Mlist) mwd[e] = bal[e] & ~m.pmask[w];
      if (lane == 0) {
        m.amask[w] = bal[e];
        m.offs[w] = ((uint32_t)__popc(bal[e]) << 16) | (uint32_t)__popc(mwd[e]);
      }
      // A missed block goes out the moment it is known, in ANY repair slot (a shared-memory ticket):
      // the repair units and the merge do not care about the order, and the ordered lists (A and M
      // as the API reports them) are written later, off the critical path.
      if ((mwd[e] >> lane) & 1u) {
        const uint32_t pos = atomicAdd(&dec[8], 1u);
        st_relaxed64(mtag + pos, ((unsigned long long)ep << 32) | (uint32_t)(i + 1));
      }
    }
  }
  tm.sync();
  if (tl && tm.tid == 0) tl[3] = gtime();
  if (Mlist) {
    const int nMq = (int)dec[8];
#pragma unroll 1
    for (int j = nMq + tm.tid; j < widthM; j += tm.nt) st_relaxed64(mtag + j, (unsigned long long)ep << 32);  // void tickets
    // the merge list, published before the ordered lists are written: the merge of the speculative
    // entries can start while the repairs are in flight
    uint32_t pk = 0;
    if (tm.wid == 0) pk = write_merge_list(a, row, nb, nMq, m, ep);
    tm.sync();
    if (tm.tid == 0) st_release64(&a.sel2[row], ((unsigned long long)ep << 32) | pk);
  }
  if (tm.wid == 0) {  // exclusive scan of the per-word counts, in block order
    uint32_t carry = 0;
#pragma unroll 1
    for (int w0 = 0; w0 < nwd; w0 += 32) {
      const int w = w0 + lane;
      const uint32_t v = w < nwd ? m.offs[w] : 0u;
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
  tm.sync();
  if (tl && tm.tid == 0) tl[4] = gtime();
  const uint32_t tot = dec[3];
#pragma unroll
  for (int e = 0; e < KB; ++e) {
    const int i = tm.tid + e * tm.nt, w = tm.wid + e * nw32;
    if (w < nwd) {
      const uint32_t off = m.offs[w];
      if ((bal[e] >> lane) & 1u) list[(off >> 16) + __popc(bal[e] & lt)] = i;
      if ((mwd[e] >> lane) & 1u) Mlist[(off & 0xffffu) + __popc(mwd[e] & lt)] = i;
      if (mask_g && lane == 0) mask_g[w] = bal[e];
    }
  }
#pragma unroll 1
  for (int j = (int)(tot >> 16) + tm.tid; j < width; j += tm.nt) list[j] = -1;
  if (Mlist)
#pragma unroll 1
    for (int j = (int)(tot & 0xffffu) + tm.tid; j < widthM; j += tm.nt) Mlist[j] = -1;
  tm.sync();
  return tot;
}

// The row's scores for the blocks this thread owns (t, t + nt, ...), polled as epoch-tagged words:
// every missing word is re-requested each round (all in flight together), the warp leaves on a vote.
__device__ __forceinline__ void poll_scores(const unsigned long long* s64, int nb, int tid, int nt, uint32_t ep,
                                            float (&x)[KB], uint32_t* err) {
  uint32_t pend = 0u;
#pragma unroll
  for (int e = 0; e < KB; ++e) {
    x[e] = 0.f;
    if (tid + e * nt < nb) pend |= 1u << e;
  }
  uint32_t it = 0;
#pragma unroll 1
  for (;;) {
    unsigned long long w[KB];
#pragma unroll
    for (int e = 0; e < KB; ++e) w[e] = (pend >> e) & 1u ? ld_relaxed64(s64 + tid + e * nt) : 0ull;
#pragma unroll
    for (int e = 0; e < KB; ++e)
      if (((pend >> e) & 1u) && (uint32_t)(w[e] >> 32) == ep) {
        x[e] = __uint_as_float((uint32_t)w[e]);
        pend &= ~(1u << e);
      }
    if (__all_sync(FULL, pend == 0u)) break;
    __nanosleep(20);
    if (++it > SPIN_LIMIT) { if ((threadIdx.x & 31) == 0) atomicExch(err, 1u); break; }
  }
}

// ---------------------------------------------------------------------------------------------
// One row job by one team (a single code path for both kinds, so the kernel holds ONE copy of the
// selection code: the instruction cache is 32 KB and this code runs once per step, on the
// critical path).
//   select(row): a2 + a5.  Before the scores exist: bitmask of the predicted set P in shared
//                memory.  After: keys -> exact K-th -> A ascending + bitmask, M = A\P, publish.
//   ema(row):    a8 + a3.  Before the scores exist: the row's (l, v) state is staged in shared
//                memory (HBM latency hidden behind the score phase).  After: Eq. 3 in
//                non-contracted fp64 (both lines use l^{t-1}; blocks scored for the first time
//                get l = IS, v = 0), Eq. 2 rounded once to fp32, the same exact
//                selection -> P = top-min(Bud, #stateful) of the NEXT step.
__device__ void run_job(const StepArgs& a, int jj, int R, const Team& tm, const TeamMem& m, const int32_t* Pcur,
                        int32_t* Pnext, uint32_t ep, unsigned long long* tl) {
  const bool is_sel = jj < R;
  const int row = is_sel ? jj : jj - R;
  const int b = row / a.Hkv;
  const int nb = max(0, min(a.MB, (seq_len(a, b) + a.bs - 1) / a.bs));
  uint32_t* dec = m.red + tm.nw * 16;
  uint32_t* ctl = a.ctl;
  const float* sc = a.scores + (size_t)row * a.MB;
  double* L = a.ema_l + (size_t)row * a.MB;
  double* V = a.ema_v + (size_t)row * a.MB;
  int np = 0, n_old = 0, n = nb;
  bool st_sm = false;
  // ---- before the scores ----
  if (is_sel) {
#pragma unroll 1
    for (int w = tm.tid; w < a.MBw; w += tm.nt) m.pmask[w] = 0u;
    if (tm.tid == 0) { dec[4] = 0u; dec[8] = 0u; }
    tm.sync();
    if (a.spec) {
      const int32_t* P = Pcur + (size_t)row * a.Bud;
      for (int j = tm.tid; j < a.Bud; j += tm.nt) {
        const int blk = __ldcg(P + j);
        const bool ok = blk >= 0 && blk < a.MB;
        m.plist[j] = ok ? blk : -1;
        if (ok) { atomicOr(&m.pmask[blk >> 5], 1u << (blk & 31)); ++np; }
      }
      np = __reduce_add_sync(FULL, np);
      if ((threadIdx.x & 31) == 0 && np) atomicAdd(&dec[4], (uint32_t)np);
    }
    tm.sync();
    np = (int)dec[4];
  } else {
    n_old = a.n_state[row];
    n = max(nb, n_old);
    st_sm = n <= m.st_cap;
    if (st_sm) {
#pragma unroll 1
      for (int i0 = tm.tid; i0 < n_old; i0 += 6 * tm.nt) {
        double x[6], y[6];
#pragma unroll
        for (int e = 0; e < 6; ++e) {
          const int i = i0 + e * tm.nt;
          x[e] = i < n_old ? L[i] : 0.0;
          y[e] = i < n_old ? V[i] : 0.0;
        }
#pragma unroll
        for (int e = 0; e < 6; ++e) {
          const int i = i0 + e * tm.nt;
          if (i < n_old) { m.Ls[i] = x[e]; m.Vs[i] = y[e]; }
        }
      }
    }
  }
  const bool in_sm = n <= m.key_cap;
  const bool fast = in_sm && n <= KB * tm.nt;  // (uniform over the team)
  const unsigned long long* s64 = a.sc64 + (size_t)row * a.MB;
  // ---- wait for the row's scores (the fast path polls the tagged score words themselves, below) ----
  if (tm.wid == 0) {  // one flag per score chunk of the row, a few per lane
    const int cprs = (a.MB + a.CR - 1) / a.CR, target = (nb + a.CR - 1) / a.CR;
    const uint32_t* f = a.sfl + (size_t)row * cprs;
    // (fast path: only the row's first chunk flag, as the sign that the scores are about to land --
    // polling 2048 tagged words per row from the start of the step would load L2 for nothing)
    wait_flags(f, fast ? min(1, target) : target, ep, &ctl[CTL_ERR]);
  }
  tm.sync();
  if (tl && tm.tid == 0) tl[8] = gtime();
  // ---- keys ----
  uint32_t kmin = 0xffffffffu, kmax = 0u;
  float* pr = a.pred + (size_t)row * a.MB;
  float xf[KB];
  if (fast) {  // every thread of the team takes part (votes inside)
    poll_scores(s64, nb, tm.tid, tm.nt, ep, xf, &ctl[CTL_ERR]);
    if (tl && tm.tid == 0) tl[8] = gtime();
  }
  if (is_sel) {
#pragma unroll 1
    for (int i0 = tm.tid; i0 < nb; i0 += KB * tm.nt) {
      float x[KB];
#pragma unroll
      for (int e = 0; e < KB; ++e) {
        const int i = i0 + e * tm.nt;
        x[e] = fast ? xf[e] : (i < nb ? __ldcg(sc + i) : 0.f);
      }
#pragma unroll
      for (int e = 0; e < KB; ++e) {
        const int i = i0 + e * tm.nt;
        if (i < nb) {
          const uint32_t key = score_key(x[e]);
          if (in_sm) m.keys[i] = key;
          kmin = min(kmin, key);
          kmax = max(kmax, key);
        }
      }
    }
  } else {
    const double alpha = a.theta[b * 3 + 0], beta = a.theta[b * 3 + 1], gamma = a.theta[b * 3 + 2];
    const double oma = __dsub_rn(1.0, alpha), omb = __dsub_rn(1.0, beta);
    if (in_sm) {  // the row's scores, every load in flight at once; each thread re-reads only what it stored
#pragma unroll 1
      for (int i0 = tm.tid; i0 < nb; i0 += KB * tm.nt) {
        float x[KB];
#pragma unroll
        for (int e = 0; e < KB; ++e) {
          const int i = i0 + e * tm.nt;
          x[e] = fast ? xf[e] : (i < nb ? __ldcg(sc + i) : 0.f);
        }
#pragma unroll
        for (int e = 0; e < KB; ++e) {
          const int i = i0 + e * tm.nt;
          if (i < nb) m.keys[i] = __float_as_uint(x[e]);
        }
      }
    }
#pragma unroll 2
    for (int i = tm.tid; i < n; i += tm.nt) {
      const bool has = i < n_old;
      double ln = 0.0, vn = 0.0;
      if (has) { ln = st_sm ? m.Ls[i] : L[i]; vn = st_sm ? m.Vs[i] : V[i]; }
      if (i < nb) {
        const double xd = (double)(in_sm ? __uint_as_float(m.keys[i]) : __ldcg(sc + i));
        if (has) {
          const double lo_ = ln;
          vn = __dadd_rn(__dmul_rn(beta, __dsub_rn(xd, lo_)), __dmul_rn(omb, vn));
          ln = __dadd_rn(__dmul_rn(alpha, xd), __dmul_rn(oma, lo_));
        } else {
          ln = xd;
          vn = 0.0;
        }
        L[i] = ln;
        V[i] = vn;
      }
      const float p = f64_to_score(__dadd_rn(ln, __dmul_rn(gamma, vn)));
      const uint32_t key = score_key(p);
      if (in_sm) m.keys[i] = key; else pr[i] = p;
      kmin = min(kmin, key);
      kmax = max(kmax, key);
    }
    tm.sync();  // n_state is read by every thread above, written below
    if (tm.tid == 0) a.n_state[row] = n;
    if (a.Bud <= 0) return;
  }
  // ---- exact selection (one call site) ----
  const int bsel = a.bud_seq[b] > 0 ? min(a.bud_seq[b] - 1, a.Bud) : a.BudSel;
  const int k = min(is_sel ? a.K : bsel, n);
  Keys ks{in_sm ? smem_u32(m.keys) : 0u, is_sel ? sc : pr};
  Thr t;
  t.key = 0u; t.idx = 0x7fffffff;  // k >= n: everything is selected
  uint32_t kreg[KB];
  if (fast) {
#pragma unroll
    for (int e = 0; e < KB; ++e) {  // each thread re-reads only what it stored
      const int i = tm.tid + e * tm.nt;
      kreg[e] = i < n ? m.keys[i] : 0u;
    }
  }
  if (k > 0 && k < n) {
    if (fast) {
      if (tl && tm.tid == 0) tl[9] = gtime();
      t = fast_kth(kreg, ks, n, k, tm, m, tl);
    } else {
      uint32_t lo, span;
      team_range(kmin, kmax, tm, m, lo, span);
      if (tl && tm.tid == 0) tl[9] = gtime();
      t = team_kth(ks, n, k, tm, m, lo, span, n);
    }
  } else {
    tm.sync();
  }
  if (tl && tm.tid == 0) tl[10] = gtime();
  int32_t* list = is_sel ? a.setA + (size_t)row * a.K : Pnext + (size_t)row * a.Bud;
  uint32_t* mask_g = is_sel ? a.maskA + (size_t)row * a.MBw : nullptr;
  int32_t* Mlist = is_sel ? a.setM + (size_t)row * a.K : nullptr;
  const uint32_t tot = fast ? fast_emit(kreg, n, k, t, tm, m, list, is_sel ? a.K : a.Bud, mask_g, Mlist, a.K,
                                            is_sel ? a.mtag + (size_t)row * a.K : nullptr, ep, a, row, nb, tl)
                            : team_emit(ks, n, k, t, tm, m, list, is_sel ? a.K : a.Bud, mask_g, Mlist, a.K);
  if (tl && tm.tid == 0) tl[11] = gtime();
  if (!is_sel) return;
  if (!fast) {  // generic path: the tagged words from the list just written (team_emit ended with a barrier)
    const int nMg = (int)(tot & 0xffffu);
    for (int j = tm.tid; j < a.K; j += tm.nt) {
      const int blk = j < nMg ? __ldcg(Mlist + j) : -1;
      st_relaxed64(a.mtag + (size_t)row * a.K + j, ((unsigned long long)ep << 32) | (uint32_t)(blk + 1));
    }
  }
  // ---- publish (select only) ----
  const int nA = (int)(tot >> 16), nM = (int)(tot & 0xffffu);
  uint32_t pkg = 0;
  if (!fast && tm.wid == 0) pkg = write_merge_list(a, row, nb, nM, m, ep);  // (the fast path wrote and published it already)
  if (tm.tid == 0) {
    a.counts[row * 3 + 0] = nA;
    a.counts[row * 3 + 1] = np;
    a.counts[row * 3 + 2] = nM;
    if (a.stats) {
      atomicAdd(&a.stats[0], (unsigned long long)nA);
      atomicAdd(&a.stats[1], (unsigned long long)(nA - nM));
      atomicAdd(&a.stats[2], (unsigned long long)nM);
      atomicAdd(&a.stats[3], (unsigned long long)np);
    }
  }
  tm.sync();  // every thread's stores (A, M, merge list, counts) are ordered before the release
  if (tm.tid == 0) {
    st_release(&a.sel[row], ep);
    if (!fast) st_release64(&a.sel2[row], ((unsigned long long)ep << 32) | pkg);
  }
}

// a7 for one (sequence, query head, 16-channel slice of d): Eq. 6-8 over the listed partial states,
// O unnormalised and one division at the end.  The warp is 8 groups of 4 lanes; a group owns every
// 8th entry and its lanes one float4 of the 64-byte slice, so a pass has 80 entries in flight (the
// whole speculative segment of a row in one round trip); the groups are folded with three shuffles.  Entries are folded speculative slots
// ascending, then repair slots ascending; a missed block takes whichever repair slot its shared-memory
// ticket gave it (warp-scheduling order), so the fp32 rounding of the repair segment can differ from run
// to run by a few ulp (tests bound it by 2e-6); any order is the same real number (Q11).
template <int D, int MSW>
__device__ void job_merge(const StepArgs& a, int b, int hq, int dq, unsigned char* buf, uint32_t ep,
                          unsigned long long* tl) {
  constexpr uint32_t REP = 0x80000000u;
  const int lane = threadIdx.x & 31;
  const int h = hq / a.G, row = b * a.Hkv + h;
  const size_t hb = (size_t)b * a.Hq + hq;
  const int E = a.Bud + a.K;
  float* ws = reinterpret_cast<float*>(buf);             // [E] m, then weights
  uint32_t* cs = reinterpret_cast<uint32_t*>(buf) + E;   // [E] slot codes (REP bit: repair buffers)
  float* ls = reinterpret_cast<float*>(buf) + 2 * E;     // [E] l
  // The row's merge list is written by select(row): slot codes, speculative slots first, as epoch-
  // tagged words; this warp polls all E of them (MERGE_END past the end) and has list and lengths in
  // one round trip once they exist.
  int n = 0, nh = 0;
  {
    const unsigned long long* m64 = a.ms64 + (size_t)row * E;
#pragma unroll 1
    for (int eb = 0; eb < E; eb += 4 * 32) {  // warp-uniform trips (votes inside)
      uint32_t c4[4] = {MERGE_END, MERGE_END, MERGE_END, MERGE_END};
      uint32_t pend = 0u, it = 0;
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (eb + lane + 32 * u < E) pend |= 1u << u;
#pragma unroll 1
      for (;;) {
        unsigned long long w[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) w[u] = (pend >> u) & 1u ? ld_relaxed64(m64 + eb + lane + 32 * u) : 0ull;
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (((pend >> u) & 1u) && (uint32_t)(w[u] >> 32) == ep) { c4[u] = (uint32_t)w[u]; pend &= ~(1u << u); }
        if (__all_sync(FULL, pend == 0u)) break;
        __nanosleep(40);
        if (++it > SPIN_LIMIT) { if (lane == 0) atomicExch(a.ctl + CTL_ERR, 1u); break; }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int e = eb + lane + 32 * u;
        const bool valid = e < E && c4[u] != MERGE_END;
        if (e < E) cs[e] = c4[u];
        n += __popc(__ballot_sync(FULL, valid));
        nh += __popc(__ballot_sync(FULL, valid && !(c4[u] & REP)));
      }
    }
    __syncwarp();
  }
  if (tl && lane == 0) tl[12] = gtime();
  // slice of msw channels: msw / 4 lanes x float4 per entry group, 128 / msw entry groups per warp
  constexpr int lpg = MSW / 4, ng = 32 / lpg;
  const int grp = lane / lpg, l8 = lane % lpg;
  const float* Os = a.O_spec + hb * a.Bud * D + dq * MSW + l8 * 4;
  const float* Or = a.O_rep + hb * a.K * D + dq * MSW + l8 * 4;
  // Two segments folded by Eq. 6-8: first the speculative entries (their units finished while
  // selection ran), then the repaired ones -- so only the few repair rows are left to fetch once
  // the last repair unit has published.  A segment is processed in trips of <= 128 entries: poll the
  // entries' tagged m words (acquire: flag and m in one), request l and the partial rows together,
  // weights from m, fold the trip into the running state.
  const unsigned long long* Ms = a.mt_spec + hb * a.Bud;
  const unsigned long long* Mr = a.mt_rep + hb * a.K;
  float mrun = -CUDART_INF_F, lrun = 0.f;
  float4 arun = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
  for (int seg = 0; seg < 2; ++seg) {
    const int sb = seg ? nh : 0, se = seg ? n : nh;
#pragma unroll 1
    for (int s0 = sb; s0 < se; s0 += 4 * 32) {  // warp-uniform trips (votes inside)
      const int s1 = min(se, s0 + 4 * 32);
      const int e0 = s0 + lane;
      uint32_t code[4];
      float me[4], le[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        code[u] = e0 + 32 * u < s1 ? cs[e0 + 32 * u] : 0u;
        me[u] = -CUDART_INF_F;
      }
      {  // wait for exactly these entries' units (over-predicted blocks that are not merged are not
         // waited for); the warp stays converged and exits on a vote
        uint32_t pend = 0u, it = 0;
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (e0 + 32 * u < s1) pend |= 1u << u;
#pragma unroll 1
        for (;;) {
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if ((pend >> u) & 1u) {
              const uint32_t j = code[u] & ~REP;
              const unsigned long long w = ld_acquire64((code[u] & REP) ? Mr + j : Ms + j);
              if ((uint32_t)(w >> 32) == ep) { me[u] = __uint_as_float((uint32_t)w); pend &= ~(1u << u); }
            }
          if (__all_sync(FULL, pend == 0u)) break;
          __nanosleep(20);
          if (++it > SPIN_LIMIT) { if (lane == 0) atomicExch(a.ctl + CTL_ERR, 1u); break; }
        }
      }
      if (tl && lane == 0) tl[13 + seg] = gtime();
      float mx = -CUDART_INF_F;
#pragma unroll
      for (int u = 0; u < 4; ++u) {  // l is requested now and used after the partial rows are in flight
        const uint32_t j = code[u] & ~REP;
        const bool on = e0 + 32 * u < s1;
        le[u] = on ? __ldcg((code[u] & REP) ? a.l_rep + hb * a.K + j : a.l_spec + hb * a.Bud + j) : 0.f;
        mx = fmaxf(mx, me[u]);
      }
#pragma unroll
      for (int off = 16; off >= 1; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, off));
      float wl[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        wl[u] = me[u] == -CUDART_INF_F ? 0.f : ex2((me[u] - mx) * LOG2E_F);
        if (e0 + 32 * u < s1) ws[e0 + 32 * u] = wl[u];
      }
      __syncwarp();
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
      for (int g0 = s0 + grp; g0 < s1; g0 += ng * 10) {  // 10 rows per lane in flight (80 entries per warp at 16 channels)
        float4 x[10];
        float w[10];
#pragma unroll
        for (int u = 0; u < 10; ++u) {
          const int e = g0 + ng * u;
          const bool on = e < s1;
          const uint32_t cd = on ? cs[e] : 0u;
          w[u] = on ? ws[e] : 0.f;
          const float* Op = (cd & REP) ? Or + (size_t)(cd & ~REP) * D : Os + (size_t)cd * D;
          x[u] = on ? __ldcg(reinterpret_cast<const float4*>(Op)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < 10; ++u) {
          acc.x = fmaf(w[u], x[u].x, acc.x); acc.y = fmaf(w[u], x[u].y, acc.y);
          acc.z = fmaf(w[u], x[u].z, acc.z); acc.w = fmaf(w[u], x[u].w, acc.w);
        }
      }
      float lsum = 0.f;
#pragma unroll
      for (int u = 0; u < 4; ++u) lsum = fmaf(wl[u], le[u], lsum);
#pragma unroll
      for (int off = 16; off >= 1; off >>= 1) lsum += __shfl_xor_sync(FULL, lsum, off);
      __syncwarp();  // ws[] of this trip is consumed
      // fold the trip into the running state (Eq. 6-8, unnormalised)
      const float mnew = fmaxf(mrun, mx);
      const float fo = mrun == -CUDART_INF_F ? 0.f : ex2((mrun - mnew) * LOG2E_F);
      const float fn = mx == -CUDART_INF_F ? 0.f : ex2((mx - mnew) * LOG2E_F);
      arun.x = fo * arun.x + fn * acc.x; arun.y = fo * arun.y + fn * acc.y;
      arun.z = fo * arun.z + fn * acc.z; arun.w = fo * arun.w + fn * acc.w;
      lrun = fo * lrun + fn * lsum;
      mrun = mnew;
    }
  }
#pragma unroll
  for (int off = lpg; off <= 16; off <<= 1) {
    arun.x += __shfl_xor_sync(FULL, arun.x, off); arun.y += __shfl_xor_sync(FULL, arun.y, off);
    arun.z += __shfl_xor_sync(FULL, arun.z, off); arun.w += __shfl_xor_sync(FULL, arun.w, off);
  }
  if (grp == 0) {
    float4 o;
    o.x = lrun > 0.f ? arun.x / lrun : 0.f; o.y = lrun > 0.f ? arun.y / lrun : 0.f;
    o.z = lrun > 0.f ? arun.z / lrun : 0.f; o.w = lrun > 0.f ? arun.w / lrun : 0.f;
    *reinterpret_cast<float4*>(a.out + hb * D + dq * MSW + l8 * 4) = o;
  }
  __syncwarp();
}

// ---------------------------------------------------------------------------------------------
template <int D, int BS>
__global__ void __launch_bounds__(32 * Tile<D, BS>::WMAX, 1) k_step(const __grid_constant__ StepArgs a) {
  constexpr int LPR = D / 8;
  const int NQ = D / a.msw;                              // merge slices per query head
  const int CR = a.CR;                                   // rows per score chunk
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  __shared__ __align__(8) unsigned long long bars_all[2 * 12];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
  const int NC = gridDim.x, NW = W * NC;
  const int per_warp = a.buf_bytes + a.scr_bytes;
  unsigned char* buf = smem_raw + (size_t)warp * per_warp;
  unsigned char* Ks = buf;
  unsigned long long* bars = bars_all + 2 * warp;
  uint32_t ph = 0;  // parity of the next tile to land in this warp's buffer
  if (lane == 0) { mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_fence_init(); }
  __syncwarp();
  // Programmatic dependent launch: let the next step's grid be scheduled now (its CTAs take the SMs
  // as ours exit and its launch latency hides behind this step), and wait for the previous step's
  // grid to have completed before the first global access.  No-ops without the launch attribute.
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");
  uint32_t* ctl = a.ctl;
  // The epoch and the prediction parity are loaded now and first USED after the warp's summary rows
  // and queries are in flight (an in-order warp stalls at the first use of a pending load).
  const uint32_t ep0 = __ldcg(ctl + CTL_EPOCH);
  const int par_raw = __ldcg(a.parity);
  const int R = a.B * a.Hkv;
  uint32_t ep;  // this launch's epoch: the value every flag of the step takes
  int par;
  const int32_t* Pcur;
  int32_t* Pnext;
  unsigned long long* tl = a.tl ? a.tl + ((size_t)blockIdx.x * W + warp) * 16 : nullptr;
  if (tl && lane == 0) { tl[0] = gtime(); tl[8] = 0; tl[9] = 0; tl[10] = 0; tl[11] = 0; tl[12] = 0; tl[13] = 0; tl[14] = 0; tl[15] = 0; }

  // Roles.  Team mode (J job CTAs at the end of the grid, one row job each): the job CTAs take no
  // score chunk (they stage P / the EMA state and then wait) and are ranked after every worker
  // warp, so speculative units land on worker CTAs first.  Warp mode (J = 0): the highest-numbered
  // warps take the row jobs after their score chunk.
  const int NWK = NC - a.J;
  const bool job_cta = (int)blockIdx.x >= NWK;
  const int gw = warp * NWK + (int)blockIdx.x;  // worker-warp id: consecutive ids sit on different SMs
  const int NWS = NWK * W;                      // warps that score
  const bool job_warp = a.J == 0 && (NW - 1 - gw) < 2 * R;

  // the unit this warp computes next: (ub, uh, ublk) with its tile in flight when `pend`
  const int U = a.spec ? R * a.Bud : 0;
  int u = gw;
  int ub = 0, uh = 0, ublk = -1, uvalid = 0, upage = 0, urow = 0, uslot = 0;
  bool urep = false, pend = false;
  int ulen = 0;
  auto unit_decode_a = [&](int unit) {  // issue the independent loads (no use of their values yet)
    uslot = unit / R; urow = unit - uslot * R;
    ub = urow / a.Hkv; uh = urow - ub * a.Hkv;
    ublk = __ldcg(Pcur + (size_t)urow * a.Bud + uslot);
    ulen = seq_len(a, ub);
  };
  auto unit_decode_b = [&]() {
    if (ublk >= a.MB) ublk = -1;
    uvalid = 0;
    if (ublk >= 0) {
      uvalid = min(BS, ulen - ublk * BS);
      upage = __ldg(a.table + (size_t)ub * a.MB + ublk);
    }
  };
  auto unit_decode = [&](int unit) { unit_decode_a(unit); unit_decode_b(); };
  const bool prefetch = !job_cta && !job_warp && u < U;

  // ---- phase 1: scores.  The warp's first speculative tile goes in flight only once its summary
  // rows have LANDED: the 25 MB of tile traffic would otherwise queue in front of the 4 MB that
  // heads the critical path.
  if (!job_cta) {
    const int cpr = (a.MB + CR - 1) / CR;  // chunks per row (static upper bound)
    const int maxr = a.buf_bytes / (LPR * 16);  // rows the staging buffer holds
#pragma unroll 1
    for (int it = gw; it < R * cpr; it += NWS) {
      const int ch = it / R, row = it - ch * R;
      const int b = row / a.Hkv, h = row - b * a.Hkv;
      const int end = min(a.MB, (ch + 1) * CR);
      int nb = 0;
#pragma unroll 1
      for (int r0 = ch * CR; r0 < end; r0 += maxr) {
        nb = score_chunk<D>(a, b, h, r0, min(end, r0 + maxr), Ks, ep0 + 1u, tl);
        if (r0 + maxr >= nb) break;
      }
      if (tl && lane == 0) tl[14] = gtime();
      if (ch * CR >= nb) continue;  // a chunk past the sequence's last block: nobody waits for it
      signal_set(&a.sfl[(size_t)row * cpr + ch], ep0 + 1u);
      if (tl && lane == 0) tl[15] = gtime();
    }
    ep = ep0 + 1u; par = par_raw & 1;
    Pcur = par ? a.P1 : a.P0; Pnext = par ? a.P0 : a.P1;
    if (prefetch) unit_decode(u);
    // No bulk tile traffic from this SM before all of its warps have published their scores: a
    // release waits for the SM's outstanding memory traffic.
    __syncthreads();
    if (prefetch && ublk >= 0) {
      // Traffic shaping: the first wave of speculative tiles is issued at the rate HBM can serve it
      // (warp gw waits gw x tile_time) instead of all at once, so the queues in front of L2 stay
      // short and the small critical-path accesses (flags, scores, lists) are not stuck behind
      // megabytes of bulk requests.  Total speculative time is unchanged: it is bandwidth-bound.
      if (a.pace_ns > 0.f) {
        const unsigned long long t_go = gtime() + (unsigned long long)((float)gw * a.pace_ns);
        while (gtime() < t_go) __nanosleep(32);
      }
      tile_load<D, BS>(Ks, bars, a, upage, uh);
      pend = true;
      if (tl && lane == 0) tl[7] = gtime();
    }
  }
  if (job_cta) {
    ep = ep0 + 1u; par = par_raw & 1;
    Pcur = par ? a.P1 : a.P0; Pnext = par ? a.P0 : a.P1;
  }
  if (tl && lane == 0) tl[1] = gtime();

  // ---- phase 2: row jobs -------------------------------------------------------------------------
  if (job_cta || job_warp) {
    Team tm;
    TeamMem m;
    uint32_t* p;
    size_t cap_bytes;
    if (job_cta) {
      tm = Team{(int)threadIdx.x, (int)blockDim.x, warp, W, true};
      p = reinterpret_cast<uint32_t*>(smem_raw);
      m.hbits = 11;
    } else {
      tm = Team{lane, 32, 0, 1, false};
      p = reinterpret_cast<uint32_t*>(buf + a.buf_bytes);
      m.hbits = 8;
    }
    m.pmask = p; p += a.MBw;
    m.amask = p; p += a.MBw;
    m.offs = p; p += a.MBw;
    m.red = p; p += tm.nw * 16 + 16;
    m.hist = p; p += 1 << m.hbits;
#pragma unroll 1
    for (int i = tm.tid; i < (1 << m.hbits); i += tm.nt) m.hist[i] = 0u;
    p += ((uintptr_t)p >> 2) & 1;  // 8-byte alignment
    m.cand = reinterpret_cast<unsigned long long*>(p); p += 2 * CAND;
    m.rk = p; p += CAND;
    for (int i = tm.tid; i < CAND; i += tm.nt) m.rk[i] = 0u;
    m.plist = reinterpret_cast<int32_t*>(p); p += a.Bud;
    unsigned char* pool;
    if (job_cta) {
      pool = reinterpret_cast<unsigned char*>(p);
      cap_bytes = (size_t)W * per_warp - (size_t)(pool - smem_raw);
    } else {
      pool = buf;
      cap_bytes = (size_t)a.buf_bytes;
    }
    pool += (16 - ((uintptr_t)pool & 15)) & 15;
    // pool: keys [cap] u32, then l [cap], v [cap] fp64 (20 bytes per block)
    const int cap = (int)((cap_bytes - 16) / 20) & ~3;
    m.keys = reinterpret_cast<uint32_t*>(pool);
    m.key_cap = cap;
    m.Ls = reinterpret_cast<double*>(pool + (size_t)cap * 4);
    m.Vs = m.Ls + cap;
    m.st_cap = cap;
    const int j0 = job_cta ? (int)blockIdx.x - NWK : NW - 1 - gw;
    const int jstep = job_cta ? a.J : NW;
#pragma unroll 1
    for (int jj = j0; jj < 2 * R; jj += jstep) {
      run_job(a, jj, R, tm, m, Pcur, Pnext, ep, tl);
      tm.sync();
    }
    tm.sync();  // the team's memory becomes per-warp tile buffers again
  }
  if (tl && lane == 0) tl[2] = gtime();

  // ---- phases 3 + 4: per-block partial states.  First this warp's share of the speculative units
  // (a4, static, the next tile is put in flight before the finished one is published), then
  // repair units (a6) claimed by ticket -> (row, slot) by whichever warp is free, each waiting
  // for select(row).  One loop, one copy of the tile code.
  if (!job_cta) {
    const int NT = R * a.K;
    bool finished = false;
    int tr = gw;  // next repair ticket of this warp
#pragma unroll 1
    for (;;) {
      if (!pend) {
        if (u < U) {
          unit_decode(u);
          if (ublk < 0) { u += NWS; continue; }
          urep = false;
        } else {
          if (tl && lane == 0 && !urep) tl[3] = gtime();
          // the next repair unit of this warp: tickets (slot-major) are dealt out statically; a
          // ticket is void when its row has fewer misses than its slot
#pragma unroll 1
          for (;;) {
            if (tr >= NT) { finished = true; break; }
            uslot = tr / R; urow = tr - uslot * R;
            tr += NWS;
            unsigned long long w = 0ull;
            if (lane == 0) {  // the ticket's own word: tag = this launch's epoch once select(row) knows M
              const unsigned long long* mp = a.mtag + (size_t)urow * a.K + uslot;
              uint32_t it = 0;
              while ((uint32_t)((w = ld_relaxed64(mp)) >> 32) != ep) {
                __nanosleep(20);
                if (++it > SPIN_LIMIT) { atomicExch(&ctl[CTL_ERR], 1u); w = (unsigned long long)ep << 32; break; }
              }
            }
            ublk = (int)__shfl_sync(FULL, (uint32_t)w, 0) - 1;
            if (tl && lane == 0 && tl[8] == 0) tl[8] = gtime();
            if (ublk >= 0) break;
          }
          if (finished) break;
          urep = true;
          ub = urow / a.Hkv; uh = urow - ub * a.Hkv;
          ulen = seq_len(a, ub);
          uvalid = min(BS, ulen - ublk * BS);
          upage = __ldg(a.table + (size_t)ub * a.MB + ublk);
          if (tl && lane == 0) tl[9] = gtime() + (unsigned long long)(upage & 0);
        }
        tile_load<D, BS>(Ks, bars, a, upage, uh);
        if (tl && lane == 0 && urep) tl[10] = gtime();
      }
      const bool patch = a.app && uvalid > 0 && ublk == (ulen - 1) / BS;
      const bool crep = urep;
      tile_compute<D, BS>(Ks, bars, ph, a, ub, uh, uvalid, crep ? a.O_rep : a.O_spec, crep ? a.mt_rep : a.mt_spec,
                          crep ? a.l_rep : a.l_spec, crep ? a.K : a.Bud, uslot,
                          patch ? a.k_new + ((size_t)ub * a.Hkv + uh) * D : nullptr,
                          patch ? a.v_new + ((size_t)ub * a.Hkv + uh) * D : nullptr, ep);
      ph ^= 1u;
      pend = false;
      if (tl && lane == 0 && crep) tl[11] = gtime();
      if (!crep) {
        u += NWS;
        if (u < U) {  // refill the buffer before publishing: the next tile's latency starts now
          unit_decode(u);
          if (ublk >= 0) { tile_load<D, BS>(Ks, bars, a, upage, uh); pend = true; }
        }
      }
    }
  }
  if (tl && lane == 0) tl[4] = gtime();

  // ---- phase 5: merge, claimed by whoever is free ------------------------------------------------
  {
    // merge items are dealt out statically to the worker warps from the top (the repair tickets went
    // to the lowest-numbered ones): they have been idle since their speculative unit, while the job
    // CTAs' warps only come free when their row job ends.  What is left over goes to the job CTAs.
    const int NT = a.B * a.Hq * NQ;
    const int njw = a.J * W;
    int t0 = gw, tstep = NW;
    if (a.J) {
      if (job_cta) { t0 = NWS + ((int)blockIdx.x - NWK) * W + warp; tstep = njw; }
      else { t0 = NWS - 1 - gw; tstep = NT; }
    }
#pragma unroll 1
    for (int t = t0; t < NT; t += tstep) {
      const int bh = t / NQ, dq = t - bh * NQ;
      const int b = bh / a.Hq, hq = bh - b * a.Hq;
      const int row = b * a.Hkv + hq / a.G;
      if (a.msw == 16) job_merge<D, 16>(a, b, hq, dq, buf, ep, tl);
      else job_merge<D, D>(a, b, hq, dq, buf, ep, tl);
    }
  }
  if (tl && lane == 0) tl[5] = gtime();

  // ---- exit: the last warp of the grid resets the step's counters and flips the parity ---------
  __syncwarp();
  uint32_t last = 0;
  if (lane == 0) {
    __threadfence();
    last = atomicAdd(&ctl[CTL_EXIT], 1u) == (uint32_t)(NW - 1);
  }
  last = __shfl_sync(FULL, last, 0);
  if (last) {
    if (a.done_host && lane == 0) {  // every warp's results are ordered before its exit ticket (gpu scope); this fence carries them to the host
      __threadfence_system();
      *reinterpret_cast<volatile uint32_t*>(a.done_host) = a.done_seq;
    }
    if (a.app)
      for (int b = lane; b < a.B; b += 32)
        if (a.seq_lens_w[b] / a.bs < a.MB) a.seq_lens_w[b] += 1;  // (a full sequence: nothing was written, the length stays, as in k_append)
    if (lane == 0) {
      ctl[CTL_EXIT] = 0u;
      ctl[CTL_EPOCH] = ep;
      *a.parity = par ^ 1;
    }
  }
}

// ---------------------------------------------------------------------------------------------
template <int D, int BS>
static cudaError_t launch_step_t(prr_ctx* c, const StepArgs& a0, cudaStream_t s) {
  using T = Tile<D, BS>;
  StepArgs a = a0;
  const int merge_bytes = (c->Bud + c->K) * 12;
  const int R = a.B * a.Hkv;
  a.buf_bytes = (std::max(T::BYTES, merge_bytes) + 15) & ~15;
  // Row jobs: a whole CTA per job when rows are few (its bookkeeping lives in the CTA's pooled
  // buffers), else one warp per job with a 256-bucket histogram in its own scratch.
  a.J = 2 * R <= c->n_sm / 4 ? 2 * R : 0;
  int W = 0, per_warp = 0;
  for (;;) {
    a.scr_bytes = (3 * a.MBw + 32 + 3 * CAND + 2 + (a.J ? 0 : 256 + c->Bud)) * 4;
    a.scr_bytes += (1024 - (a.buf_bytes + a.scr_bytes) % 1024) % 1024;  // tile buffers stay 1024-byte aligned (swizzle atom)
    per_warp = a.buf_bytes + a.scr_bytes;
    W = std::min(T::WMAX, (c->smem_optin - 1024) / per_warp);
    if (W < 1) return cudaErrorInvalidConfiguration;
    const size_t team_words = (size_t)3 * a.MBw + W * 16 + 16 + 2048 + 3 * CAND + 2 + 64 + c->Bud;
    if (a.J && team_words * 4 > (size_t)W * per_warp) { a.J = 0; continue; }
    break;
  }
  if (a.J) {  // worker CTAs: enough warps for one wave of speculative units; the rest also merge
    const int U = a.spec ? R * a.Bud : 0;
    a.J = std::max(a.J, std::min(c->n_sm - (U + W - 1) / W, c->n_sm / 4));
  }
  {
    const long long mw = (long long)W * (c->n_sm - a.J);  // warps that merge (all of them in warp mode)
    a.msw = (long long)a.B * a.Hq * (D / 16) <= mw ? 16 : D;  // 16-channel slices when every merge warp gets at most one
  }
  const size_t smem = (size_t)W * per_warp;
  {  // score chunk: one per scoring warp (job CTAs do not score), so every warp's summary loads are one batch
    const int RW = 32 / (D / 8);
    const long long rows = (long long)R * a.MB, NWS = (long long)W * (c->n_sm - a.J);
    a.CR = (int)((rows + NWS - 1) / NWS);
    if (a.CR < 2 * RW) a.CR = 2 * RW;
  }
  bool& attr_set = c->coop_attr[(D == 128 ? 0 : 4) + (BS == 64 ? 0 : BS == 32 ? 1 : BS == 16 ? 2 : 3)];
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute((const void*)k_step<D, BS>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin - 1024);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(c->n_sm);
  cfg.blockDim = dim3(32 * W);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeCooperative;
  at[0].val.cooperative = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = c->pdl ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, k_step<D, BS>, a);
}

// Tensor map of a K or V page pool for the copy engine: bf16 [rows, d] with rows = page * Hkv * bs
// (the library is not told n_pages; tile coordinates are int32, so the row extent is 2^31), box =
// [bs rows, 64 channels = 128 bytes], 128-byte swizzle.  Encoded on the host, cached per pointer.
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
static int page_map(prr_ctx* c, const void* base, CUtensorMap* out) {
  static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap is 128 bytes");
  const void* key = reinterpret_cast<const void*>(reinterpret_cast<uintptr_t>(base) | (uintptr_t)(c->bs / 16 - 1));  // (16-byte aligned base)
  auto it = c->tmaps.find(key);
  if (it == c->tmaps.end()) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return (int)cudaErrorNotSupported;
    alignas(64) CUtensorMap m;
    const cuuint64_t dims[2] = {(cuuint64_t)c->D, (cuuint64_t)1 << 31};
    const cuuint64_t strides[1] = {(cuuint64_t)c->D * 2};
    const cuuint32_t box[2] = {64u, (cuuint32_t)c->bs};
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

static int launch_step(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries, float* out,
                       int spec, cudaStream_t s, const void* k_new, const void* v_new) {
  const size_t r = (size_t)kv->layer * c->maxB * c->Hkv;
  StepArgs a{};
  if (int e = page_map(c, kv->k_pages, &a.mapK)) return e;
  if (int e = page_map(c, kv->v_pages, &a.mapV)) return e;
  a.kp = (const uint16_t*)kv->k_pages; a.vp = (const uint16_t*)kv->v_pages;
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
  a.maskA = c->maskA; a.pred = c->pred; a.mtag = c->mtag; a.sc64 = c->sc64; a.ms64 = c->ms64; a.msrc = (uint32_t*)c->merge_src; a.mn = c->merge_n;
  a.O_spec = c->O_spec; a.m_spec = c->m_spec; a.l_spec = c->l_spec;
  a.O_rep = c->O_rep; a.m_rep = c->m_rep; a.l_rep = c->l_rep;
  a.mt_spec = c->mt_spec; a.mt_rep = c->mt_rep;
  a.ctl = c->ctl; a.stats = c->stats;
  {
    const size_t rm = (size_t)c->maxB * c->Hkv;
    const size_t rme = (rm + 1) & ~(size_t)1;  // sel2 is 64-bit: keep it 8-byte aligned
    a.sel = c->ctl + CTL_HDR; a.sel2 = (unsigned long long*)(a.sel + rme); a.ufs = a.sel + rme + 2 * rm; a.ufr = a.ufs + rm * c->Bud; a.sfl = a.ufr + rm * c->K;
  } a.tl = c->tl_on ? c->tl : nullptr;
  a.B = kv->batch; a.Hq = c->Hq; a.Hkv = c->Hkv; a.G = c->G; a.MB = c->MB; a.MBw = (c->MB + 31) / 32;
  a.bs = c->bs; a.K = c->K; a.Bud = c->Bud; a.BudSel = c->bud_eff[kv->layer]; a.Rmax = c->maxB * c->Hkv;
  a.bud_seq = c->bud_seq + (size_t)kv->layer * c->maxB;
  a.retain = c->lay.overpredict_policy == PRR_RETAIN;
  a.spec = (spec && c->Bud > 0) ? 1 : 0;
  a.scale = c->sm_scale; a.score_c = c->score_c;
  // ns per speculative tile at the rate HBM can serve (0.8 x memory clock x bus width, from the device
  // attributes); PRR_OPT_PACE scales it in percent, 0 disables
  a.pace_ns = (float)c->pace_pct * 0.01f * (float)(2.0 * c->bs * c->D * 2.0) / c->hbm_gbs_est;
  cudaError_t e = cudaErrorInvalidValue;
#define PRR_CASE(DD, BB) if (c->D == DD && c->bs == BB) e = launch_step_t<DD, BB>(c, a, s);
  PRR_CASE(128, 64) PRR_CASE(128, 32) PRR_CASE(128, 16) PRR_CASE(128, 128)
  PRR_CASE(64, 64) PRR_CASE(64, 32) PRR_CASE(64, 16) PRR_CASE(64, 128)
#undef PRR_CASE
  c->launches++;
  return e == cudaSuccess ? 0 : (int)e;
}

}  // namespace persist

int launch_step_persist(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries, float* out,
                        int spec, cudaStream_t s, const void* k_new, const void* v_new) {
  return persist::launch_step(c, kv, q, summaries, out, spec, s, k_new, v_new);
}

}  // namespace prr
