// fp8 (e4m3) KV blocks with per-block power-of-two scales (PAPER.md:319 names fp8 as future work; the
// format is this build's reading): OCP e4m3 codes, ONE scale 2^e per (page, KV head)
// for K and one for V, e the smallest integer with amax <= 448 * 2^e, codes = RNE(x / 2^e) saturated.
// A power-of-two scale makes x / 2^e and code * 2^e exact, so the e4m3 rounding is the only one and the
// dequantised tile is a bf16 tile: k_partial<.., FP8> (k_attn.cu) moves HALF the bytes from HBM, widens the
// codes to bf16 in shared memory (exact) and then runs the same mma.sync arithmetic, so its partial
// states are the bits k_partial produces on the dequantised cache.
#include <cuda_fp8.h>
#include <math_constants.h>

#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {


// e4m3 code -> bf16 bits of code * 2^e (exact: 4 significant bits; |e| is far inside bf16's range)
__device__ __forceinline__ uint16_t e4m3_to_bf16_scaled(uint32_t code, float scale) {
  const __half_raw hr = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)code, __NV_E4M3);  // exact in fp16
  const float f = __half2float(__half(hr)) * scale;                                    // exact: power-of-two scale
  return (uint16_t)(__float_as_uint(f) >> 16);                                         // exact: the low 16 bits are zero
}

// One CTA per (logical block, KV head, sequence); 128 threads.  amax over the VALID tokens (exact: a max
// of bf16 magnitudes), e from its exponent and significand, codes by the RNE conversion of the exact
// quotient; token slots past the length get code 0.
__global__ void __launch_bounds__(128)
k_quantize_fp8(const uint16_t* __restrict__ pages, const int32_t* __restrict__ table, const int32_t* __restrict__ seq_lens,
               uint8_t* __restrict__ codes, float* __restrict__ scales, int Hkv, int bs, int D, int MB) {
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z, tid = threadIdx.x;
  const int len = seq_lens[b];
  const int nb = (len + bs - 1) / bs;
  if (i >= nb) return;
  const int n_i = min(bs, len - i * bs);
  const size_t page = (size_t)table[(size_t)b * MB + i];
  const size_t base = ((page * Hkv + h) * bs) * (size_t)D;
  __shared__ uint32_t red[4];
  uint32_t am = 0u;  // magnitude bits of a bf16 compare like integers
  for (int j = tid; j < n_i * D; j += 128) am = max(am, (uint32_t)(pages[base + j] & 0x7fffu));
  am = __reduce_max_sync(FULL, am);
  if ((tid & 31) == 0) red[tid >> 5] = am;
  __syncthreads();
  am = max(max(red[0], red[1]), max(red[2], red[3]));
  // amax = m 2^x with 0.5 <= m < 1: e = x - 9 if m <= 0.875 else x - 8 (448 = 0.875 * 2^9); amax = 0 -> e = 0
  int e = 0;
  if (am != 0u) {
    const float amax = __uint_as_float(am << 16);
    int x;
    const float m = frexpf(amax, &x);
    e = m <= 0.875f ? x - 9 : x - 8;
  }
  const float inv = ldexpf(1.f, -e);
  if (tid == 0) scales[page * Hkv + h] = ldexpf(1.f, e);
  for (int j = tid; j < bs * D; j += 128) {
    uint8_t c = 0;
    if (j < n_i * D) {
      const float x = __uint_as_float((uint32_t)pages[base + j] << 16) * inv;  // exact (power of two), |x| <= 448
      c = (uint8_t)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E4M3);        // round to nearest even
    }
    codes[base + j] = c;
  }
}

// Mean-key summaries of an fp8 cache: bf16_rne(exact mean of the dequantised valid tokens) (Q2).  A code
// times a power of two is exact in fp64 and so is the sum of <= 128 of them (<= 4 + 17 + 7 bits).
__global__ void k_build_summaries_fp8(const uint8_t* __restrict__ kp, const float* __restrict__ kscale,
                                      const int32_t* __restrict__ table, const int32_t* __restrict__ seq_lens,
                                      uint16_t* __restrict__ summ, double* __restrict__ open_sum, int Hkv, int bs,
                                      int D, int MB) {
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z, c = threadIdx.x;
  const int len = seq_lens[b];
  const int nb = (len + bs - 1) / bs;
  if (i >= nb) return;
  const int n_i = min(bs, len - i * bs);
  const size_t page = (size_t)table[(size_t)b * MB + i];
  const float sc = kscale[page * Hkv + h];
  const uint8_t* src = kp + ((page * Hkv + h) * bs) * (size_t)D + c;
  double s = 0.0;
  for (int t = 0; t < n_i; ++t) s += bf16_to_f64(e4m3_to_bf16_scaled(src[(size_t)t * D], sc));
  summ[(((size_t)b * Hkv + h) * MB + i) * D + c] = f64_to_bf16_rne(__ddiv_rn(s, (double)n_i));
  if (i == nb - 1) open_sum[((size_t)b * Hkv + h) * D + c] = s;
}

void launch_quantize_fp8(prr_ctx* c, const prr_paged_kv* kv, void* k8, void* v8, float* kscale, float* vscale, cudaStream_t s) {
  dim3 grid(c->MB, c->Hkv, kv->batch);
  k_quantize_fp8<<<grid, 128, 0, s>>>((const uint16_t*)kv->k_pages, kv->block_table, kv->seq_lens, (uint8_t*)k8, kscale,
                                      c->Hkv, c->bs, c->D, c->MB);
  k_quantize_fp8<<<grid, 128, 0, s>>>((const uint16_t*)kv->v_pages, kv->block_table, kv->seq_lens, (uint8_t*)v8, vscale,
                                      c->Hkv, c->bs, c->D, c->MB);
  c->launches += 2;
}

void launch_build_summaries_fp8(prr_ctx* c, const prr_paged_kv* kv, void* summaries, cudaStream_t s) {
  dim3 grid(c->MB, c->Hkv, kv->batch);
  double* os = c->open_sum + (size_t)kv->layer * c->maxB * c->Hkv * c->D;
  k_build_summaries_fp8<<<grid, c->D, 0, s>>>((const uint8_t*)kv->k_pages, c->kscale[kv->layer], kv->block_table,
                                              kv->seq_lens, (uint16_t*)summaries, os, c->Hkv, c->bs, c->D, c->MB);
  c->launches++;
}

}  // namespace prr
