// Device-side building blocks shared by the PRR kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace prr {

constexpr unsigned FULL = 0xffffffffu;

// ---------------------------------------------------------------------------------------------
// number formats
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float bf16_lo(uint32_t x) { return __uint_as_float(x << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t x) { return __uint_as_float(x & 0xffff0000u); }
__device__ __forceinline__ double bf16_to_f64(uint16_t b) {
  return (double)__uint_as_float(((uint32_t)b) << 16);
}

// One round-to-nearest-even from fp64 to bf16 (no double rounding through fp32): truncate to
// fp32, then round the 16 dropped bits with the fp64 remainder as the sticky bit.
__device__ __forceinline__ uint16_t f64_to_bf16_rne(double x) {
  float f = __double2float_rz(x);
  uint32_t u = __float_as_uint(f);
  bool sticky = ((double)f != x);
  uint32_t low = u & 0xffffu, hi = u >> 16;
  bool up = (low > 0x8000u) || (low == 0x8000u && (sticky || (hi & 1u)));
  return (uint16_t)(hi + (up ? 1u : 0u));
}

// fp64 -> fp32 (one RNE), -0 canonicalised to +0 (Q4).
__device__ __forceinline__ float f64_to_score(double x) {
  float f = __double2float_rn(x);
  return f == 0.0f ? 0.0f : f;
}

// Order-preserving fp32 -> uint32 key: larger value <=> larger key.  +-0 share one key; NaN
// (never produced by the library) sorts below -inf.
__device__ __forceinline__ uint32_t score_key(float f) {
  if (f != f) return 0u;
  if (f == 0.0f) return 0x80000000u;
  uint32_t u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// ---------------------------------------------------------------------------------------------
// block-wide exclusive scan of a 64-bit packed counter (NT threads, NT % 32 == 0, NT <= 1024)
// ---------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ unsigned long long block_excl_scan(unsigned long long x,
                                                              unsigned long long* warp_tot,
                                                              unsigned long long* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned long long incl = x;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    unsigned long long t = __shfl_up_sync(FULL, incl, off);
    if (lane >= off) incl += t;
  }
  if (lane == 31) warp_tot[warp] = incl;
  __syncthreads();
  unsigned long long base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < NT / 32; ++w) {
    unsigned long long t = warp_tot[w];
    if (w < warp) base += t;
    tot += t;
  }
  __syncthreads();  // warp_tot may be reused by the caller
  if (total) *total = tot;
  return base + incl - x;
}

// ---------------------------------------------------------------------------------------------
// Radix select over uint32 keys held in shared memory: the threshold T = k-th largest key and
// `need` = how many keys equal to T belong to the top-k (the lowest-indexed ones).  1 <= k <= n.
// hist: 256 counters, ctl: 2 words.  Integer-only, so the result is exact and order-independent.
// ---------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ void radix_select(const uint32_t* keys, int n, int k, uint32_t* hist,
                                             uint32_t* ctl, uint32_t& T, int& need) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t prefix = 0, mask = 0;
  int remaining = k;
#pragma unroll 1
  for (int shift = 24; shift >= 0; shift -= 8) {
    for (int i = tid; i < 256; i += NT) hist[i] = 0;
    __syncthreads();
    for (int i = tid; i < n; i += NT) {
      uint32_t key = keys[i];
      if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
    }
    __syncthreads();
    if (warp == 0) {
      int c[8], sum = 0;
#pragma unroll
      for (int j = 0; j < 8; ++j) { c[j] = (int)hist[lane * 8 + j]; sum += c[j]; }
      int suf = sum;  // keys in buckets of lanes >= this one
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        int t = __shfl_down_sync(FULL, suf, off);
        if (lane + off < 32) suf += t;
      }
      int above = suf - sum;
      if (above < remaining && remaining <= suf) {
        int acc = above;
#pragma unroll
        for (int j = 7; j >= 0; --j) {
          if (acc + c[j] >= remaining) { ctl[0] = (uint32_t)(lane * 8 + j); ctl[1] = (uint32_t)(remaining - acc); break; }
          acc += c[j];
        }
      }
    }
    __syncthreads();
    prefix |= ctl[0] << shift;
    mask |= 255u << shift;
    remaining = (int)ctl[1];
  }
  T = prefix;
  need = remaining;
  __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// Ordered selection: element i is selected iff key > T, or key == T and it is among the `need`
// lowest-indexed keys equal to T.  Writes the selected indices ascending to list_out (if
// non-null) and sets their bits in `mask_words` (shared, pre-zeroed, if non-null).  Returns the
// number selected (same in every thread).  scan_tmp: 33 x u64 of shared scratch.
// ---------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ int ordered_select(const uint32_t* keys, int n, uint32_t T, int need,
                                              int* list_out, uint32_t* mask_words,
                                              unsigned long long* scan_tmp) {
  const int tid = threadIdx.x;
  const int per = (n + NT - 1) / NT;
  const int i0 = min(n, tid * per), i1 = min(n, i0 + per);
  unsigned gt = 0, eq = 0;
  for (int i = i0; i < i1; ++i) {
    uint32_t key = keys[i];
    gt += key > T;
    eq += key == T;
  }
  unsigned long long tot;
  unsigned long long ex = block_excl_scan<NT>(((unsigned long long)gt << 32) | eq, scan_tmp, &tot);
  unsigned gt_before = (unsigned)(ex >> 32), eq_before = (unsigned)(ex & 0xffffffffu);
  unsigned pos = gt_before + min(eq_before, (unsigned)need);
  unsigned eq_rank = eq_before;
  for (int i = i0; i < i1; ++i) {
    uint32_t key = keys[i];
    bool sel = key > T;
    if (key == T) { sel = eq_rank < (unsigned)need; ++eq_rank; }
    if (sel) {
      if (list_out) list_out[pos] = i;
      if (mask_words) atomicOr(&mask_words[i >> 5], 1u << (i & 31));
      ++pos;
    }
  }
  return (int)(tot >> 32) + min((int)(tot & 0xffffffffu), need);
}

// ---------------------------------------------------------------------------------------------
// async copy / tensor-core primitives
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ void ldmatrix_x4(uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3,
                                            const void* smem) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(smem_u32(smem)));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t& r0, uint32_t& r1, uint32_t& r2,
                                                  uint32_t& r3, const void* smem) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(smem_u32(smem)));
}
// D(16x8,f32) += A(16x16,bf16,row) * B(16x8,bf16,col)
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0,
                                               uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
      "{%0,%1,%2,%3};\n"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// two fp32 -> packed bf16x2 (lo in the low half), round to nearest even
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;\n" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;\n" : "=f"(y) : "f"(x));
  return y;
}

// ---------------------------------------------------------------------------------------------
// mbarrier + TMA (cp.async.bulk.tensor) primitives: the K/V tiles of the fused step are fetched by
// the copy engine, so the bulk traffic does not queue in the SM's load/store pipe in front of the
// small critical-path accesses (scores, counters, lists).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long* bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }\n"
      : "=r"(done)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return done != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// generic-proxy accesses to shared memory before this point are ordered before later async-proxy
// (TMA) accesses to it
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
// 2-D tiled tensor-map load: box at (x = innermost coordinate, y) -> dense (swizzled) shared memory
__device__ __forceinline__ void tma_load_2d(void* dst, const void* tmap, int x, int y, unsigned long long* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
      ::"r"(smem_u32(dst)), "l"(tmap), "r"(x), "r"(y), "r"(smem_u32(bar))
      : "memory");
}

}  // namespace prr
