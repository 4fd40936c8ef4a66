// a4 / a6 per-block partial attention states and a7 the merge (Eq. 6-8).
//
// k_partial: one CTA per (list slot, KV head, sequence).  The block's K and V tiles
// (block_size x head_dim bf16, contiguous in the paged cache) are staged into shared memory with
// 16-byte cp.async in two commit groups, so the QK^T pass starts while V is still in flight.  Each
// warp owns 16 tokens: S = Q K^T on mma.sync m16n8k16 (the G <= 16 query heads of the group are
// the M rows of the tile, zero padded), block-local max / sum with quad shuffles, P V on the same
// instruction, then a shared-memory combine across the block's warps.  The state is written
// relative to the BLOCK-LOCAL maximum, so a block's partial is the same bits whether it was
// computed speculatively, by the repair launch, or by the sequential baseline.
//
// k_merge: one CTA per (query head, sequence): folds the listed partial states, in ascending
// block order, with the log-sum-exp rescaling of Eq. 6-8 (written with O unnormalised and a
// single division at the end), so P\A drops out (or is retained) by simply not being listed.
#include <cuda_fp8.h>
#include <math_constants.h>

#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {

constexpr float LOG2E = 1.4426950408889634f;

// FP8: kp / vp hold e4m3 codes (one byte per element, same page layout)
// and kscale / vscale [n_pages, Hkv] their power-of-two scales.  The codes are staged raw (half the bytes
// from HBM), widened to bf16 in shared memory (code * 2^e is exact in bf16), and everything after that is
// the bf16 kernel: the partial states are the bits the bf16 kernel produces on the dequantised cache.

// The raw codes of a tile land in the TAIL of the tile's own bf16 region (BS * D bytes of its BS * LD * 2) and are
// widened in place: every thread first reads all of its chunks into registers, the block synchronises, then the
// bf16 rows are written -- so the fp8 kernel needs no more shared memory (and runs at the occupancy) of the bf16 one.
template <int D, int BS>
__device__ __forceinline__ void widen_fp8_tile(uint16_t* tile, float sc) {
  constexpr int NT = 2 * BS, LD = D + 8, NCH = (BS * D / 16) / NT;  // chunks of 16 codes per thread
  const unsigned char* raw = reinterpret_cast<const unsigned char*>(tile) + (size_t)BS * LD * 2 - (size_t)BS * D;
  uint4 v[NCH];
#pragma unroll
  for (int i = 0; i < NCH; ++i) v[i] = *reinterpret_cast<const uint4*>(raw + (size_t)(threadIdx.x + i * NT) * 16);
  __syncthreads();
#pragma unroll
  for (int i = 0; i < NCH; ++i) {
    const int c = threadIdx.x + i * NT, row = (c * 16) / D, col = (c * 16) % D;
    const uint32_t w[4] = {v[i].x, v[i].y, v[i].z, v[i].w};
    uint32_t o[8];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {  // two codes per conversion instruction (cvt.rn.f16x2.e4m3x2), exact
        const __half2_raw h2 = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)((w[j] >> (16 * e)) & 0xffffu), __NV_E4M3);
        const float2 f = __half22float2(__half2(h2));
        // code * 2^e is exact in fp32 and its low 16 bits are zero: the bf16 pair is the two high halves
        o[2 * j + e] = __byte_perm(__float_as_uint(f.x * sc), __float_as_uint(f.y * sc), 0x7632);
      }
    }
    uint4* d = reinterpret_cast<uint4*>(tile + row * LD + col);
    d[0] = make_uint4(o[0], o[1], o[2], o[3]);
    d[1] = make_uint4(o[4], o[5], o[6], o[7]);
  }
}

template <int D, int BS, bool FP8>
__global__ void __launch_bounds__(2 * BS)
k_partial(const uint16_t* __restrict__ kp, const uint16_t* __restrict__ vp,
          const int32_t* __restrict__ table, const int32_t* __restrict__ seq_lens,
          const uint16_t* __restrict__ q, const int32_t* __restrict__ list, int width,
          float* __restrict__ O, float* __restrict__ Mo, float* __restrict__ Lo, int Hq, int Hkv,
          int G, int MB, float scale, const float* __restrict__ kscale, const float* __restrict__ vscale) {
  constexpr int NT = 2 * BS;   // threads
  constexpr int TW = BS / 16;  // warps, 16 tokens each
  constexpr int LD = D + 8;    // padded row stride (elements): ldmatrix conflict-free
  constexpr int CH = D / 8;    // 16-byte chunks per row
  const int slot = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int blk = list[((size_t)b * Hkv + h) * width + slot];
  if (blk < 0) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint16_t* Ks = reinterpret_cast<uint16_t*>(smem_raw);
  uint16_t* Vs = Ks + BS * LD;
  __shared__ float mw[TW * 16], lw[TW * 16];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int valid = min(BS, seq_lens[b] - blk * BS);
  const size_t page = (size_t)table[(size_t)b * MB + blk];
  const uint16_t* gK = kp + ((page * Hkv + h) * BS) * (size_t)D;
  const uint16_t* gV = vp + ((page * Hkv + h) * BS) * (size_t)D;
  // FP8 only: the raw codes land in the tail of each tile's own region (widen_fp8_tile)
  unsigned char* rawK = reinterpret_cast<unsigned char*>(Ks) + (size_t)BS * LD * 2 - (size_t)BS * D;
  unsigned char* rawV = reinterpret_cast<unsigned char*>(Vs) + (size_t)BS * LD * 2 - (size_t)BS * D;

  if constexpr (FP8) {
    const unsigned char* gK8 = reinterpret_cast<const unsigned char*>(kp) + ((page * Hkv + h) * BS) * (size_t)D;
    const unsigned char* gV8 = reinterpret_cast<const unsigned char*>(vp) + ((page * Hkv + h) * BS) * (size_t)D;
    for (int c = tid; c < BS * D / 16; c += NT) {
      if ((c * 16) / D < valid) cp_async16(rawK + c * 16, gK8 + c * 16);
      else *reinterpret_cast<uint4*>(rawK + c * 16) = make_uint4(0, 0, 0, 0);
    }
    cp_async_commit();
    for (int c = tid; c < BS * D / 16; c += NT) {
      if ((c * 16) / D < valid) cp_async16(rawV + c * 16, gV8 + c * 16);
      else *reinterpret_cast<uint4*>(rawV + c * 16) = make_uint4(0, 0, 0, 0);
    }
    cp_async_commit();
  } else {
#pragma unroll
  for (int i = 0; i < (BS * CH) / NT; ++i) {
    const int c = tid + i * NT, row = c / CH, col = c % CH;
    uint16_t* dst = Ks + row * LD + col * 8;
    if (row < valid) cp_async16(dst, gK + row * D + col * 8);
    else *reinterpret_cast<uint4*>(dst) = make_uint4(0, 0, 0, 0);
  }
  cp_async_commit();
#pragma unroll
  for (int i = 0; i < (BS * CH) / NT; ++i) {
    const int c = tid + i * NT, row = c / CH, col = c % CH;
    uint16_t* dst = Vs + row * LD + col * 8;
    if (row < valid) cp_async16(dst, gV + row * D + col * 8);
    else *reinterpret_cast<uint4*>(dst) = make_uint4(0, 0, 0, 0);
  }
  cp_async_commit();
  }

  // Q fragments: A operand rows = query heads of the group (rows >= G are zero)
  const int r0 = lane >> 2, tq = lane & 3;
  uint32_t qa[D / 16][4];
  {
    const uint16_t* qb = q + ((size_t)b * Hq + (size_t)h * G) * D;
    const bool v0 = r0 < G, v1 = r0 + 8 < G;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
      const int col = ks * 16 + tq * 2;
      qa[ks][0] = v0 ? *reinterpret_cast<const uint32_t*>(qb + r0 * D + col) : 0u;
      qa[ks][1] = v1 ? *reinterpret_cast<const uint32_t*>(qb + (r0 + 8) * D + col) : 0u;
      qa[ks][2] = v0 ? *reinterpret_cast<const uint32_t*>(qb + r0 * D + col + 8) : 0u;
      qa[ks][3] = v1 ? *reinterpret_cast<const uint32_t*>(qb + (r0 + 8) * D + col + 8) : 0u;
    }
  }

  cp_async_wait<1>();
  __syncthreads();
  if constexpr (FP8) {
    widen_fp8_tile<D, BS>(Ks, kscale[page * Hkv + h]);
    __syncthreads();
  }

  // S = Q K^T for tokens [16*warp, 16*warp+16): two 8-token n-tiles
  const int tok0 = warp * 16;
  const int mat = lane >> 3, rr = lane & 7;
  float s[2][4];
#pragma unroll
  for (int nt = 0; nt < 2; ++nt)
#pragma unroll
    for (int e = 0; e < 4; ++e) s[nt][e] = 0.f;
#pragma unroll
  for (int k2 = 0; k2 < D / 32; ++k2) {
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      uint32_t b0, b1, b2, b3;
      ldmatrix_x4(b0, b1, b2, b3, Ks + (tok0 + nt * 8 + rr) * LD + k2 * 32 + mat * 8);
      mma_bf16_16816(s[nt], qa[2 * k2], b0, b1);
      mma_bf16_16816(s[nt], qa[2 * k2 + 1], b2, b3);
    }
  }
  // mask, block-local (here: warp-local) max and sum; rows r0 (e = 0,1) and r0+8 (e = 2,3)
  float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
#pragma unroll
  for (int nt = 0; nt < 2; ++nt)
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
  const float m0 = mx0 * scale, m1 = mx1 * scale;  // natural-log units of the scaled logit
  const float sl2 = scale * LOG2E;
  const float off0 = mx0 == -CUDART_INF_F ? 0.f : m0 * LOG2E;
  const float off1 = mx1 == -CUDART_INF_F ? 0.f : m1 * LOG2E;
  // P is fed to the tensor core as a two-term bf16 split (hi + lo), so the PV product keeps
  // ~16 significant bits of the fp32 probabilities instead of bf16's 8.
  uint32_t pa[4], pb[4];
  float l0 = 0.f, l1 = 0.f;
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    const float p0 = ex2(fmaf(s[nt][0], sl2, -off0)), p1 = ex2(fmaf(s[nt][1], sl2, -off0));
    const float p2 = ex2(fmaf(s[nt][2], sl2, -off1)), p3 = ex2(fmaf(s[nt][3], sl2, -off1));
    const uint32_t h01 = pack_bf16x2(p0, p1), h23 = pack_bf16x2(p2, p3);
    pa[nt * 2 + 0] = h01;  // (row r0,   tokens nt*8 + 2tq..)
    pa[nt * 2 + 1] = h23;  // (row r0+8, tokens nt*8 + 2tq..)
    pb[nt * 2 + 0] = pack_bf16x2(p0 - bf16_lo(h01), p1 - bf16_hi(h01));
    pb[nt * 2 + 1] = pack_bf16x2(p2 - bf16_lo(h23), p3 - bf16_hi(h23));
    l0 += p0 + p1;
    l1 += p2 + p3;
  }
  l0 += __shfl_xor_sync(FULL, l0, 1);
  l0 += __shfl_xor_sync(FULL, l0, 2);
  l1 += __shfl_xor_sync(FULL, l1, 1);
  l1 += __shfl_xor_sync(FULL, l1, 2);

  cp_async_wait<0>();
  __syncthreads();
  if constexpr (FP8) {
    widen_fp8_tile<D, BS>(Vs, vscale[page * Hkv + h]);
    __syncthreads();
  }

  // O_w = P V over this warp's 16 tokens
  float o[D / 8][4];
#pragma unroll
  for (int dt = 0; dt < D / 8; ++dt)
#pragma unroll
    for (int e = 0; e < 4; ++e) o[dt][e] = 0.f;
#pragma unroll
  for (int d2 = 0; d2 < D / 16; ++d2) {
    uint32_t b0, b1, b2, b3;
    ldmatrix_x4_trans(b0, b1, b2, b3, Vs + (tok0 + (mat & 1) * 8 + rr) * LD + d2 * 16 + (mat >> 1) * 8);
    mma_bf16_16816(o[2 * d2], pa, b0, b1);
    mma_bf16_16816(o[2 * d2], pb, b0, b1);
    mma_bf16_16816(o[2 * d2 + 1], pa, b2, b3);
    mma_bf16_16816(o[2 * d2 + 1], pb, b2, b3);
  }

  // combine the TW warps through shared memory (aliases the K/V tiles)
  __syncthreads();
  float* Ow = reinterpret_cast<float*>(smem_raw);  // [TW][16][LD] floats = BS*(D+8)*4 bytes
  if (r0 < G) {
#pragma unroll
    for (int dt = 0; dt < D / 8; ++dt)
      *reinterpret_cast<float2*>(Ow + (warp * 16 + r0) * LD + dt * 8 + tq * 2) = make_float2(o[dt][0], o[dt][1]);
    if (tq == 0) { mw[warp * 16 + r0] = m0; lw[warp * 16 + r0] = l0; }
  }
  if (r0 + 8 < G) {
#pragma unroll
    for (int dt = 0; dt < D / 8; ++dt)
      *reinterpret_cast<float2*>(Ow + (warp * 16 + r0 + 8) * LD + dt * 8 + tq * 2) = make_float2(o[dt][2], o[dt][3]);
    if (tq == 0) { mw[warp * 16 + r0 + 8] = m1; lw[warp * 16 + r0 + 8] = l1; }
  }
  __syncthreads();
  for (int idx = tid; idx < G * D; idx += NT) {
    const int row = idx / D, c = idx - row * D;
    float m = -CUDART_INF_F;
#pragma unroll
    for (int w = 0; w < TW; ++w) m = fmaxf(m, mw[w * 16 + row]);
    float acc = 0.f, lsum = 0.f;
#pragma unroll
    for (int w = 0; w < TW; ++w) {
      const float mwv = mw[w * 16 + row];
      const float f = mwv == -CUDART_INF_F ? 0.f : ex2((mwv - m) * LOG2E);
      acc = fmaf(f, Ow[(w * 16 + row) * LD + c], acc);
      lsum = fmaf(f, lw[w * 16 + row], lsum);
    }
    const size_t st = ((size_t)b * Hq + (size_t)h * G + row) * width + slot;
    O[st * D + c] = acc;
    if (c == 0) { Mo[st] = m; Lo[st] = lsum; }
  }
}

// ---------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(4 * D)
k_merge(const int32_t* __restrict__ merge_src, const int32_t* __restrict__ merge_n, int src_stride,
        const float* __restrict__ O_spec, const float* __restrict__ m_spec,
        const float* __restrict__ l_spec, int w_spec, const float* __restrict__ O_rep,
        const float* __restrict__ m_rep, const float* __restrict__ l_rep, int w_rep, int split,
        float* __restrict__ out, float* __restrict__ m_out, float* __restrict__ l_out, int Hq,
        int Hkv, int G) {
  constexpr int NT = 4 * D;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* ws = reinterpret_cast<float*>(smem_raw);       // [src_stride] weights
  int32_t* cs = reinterpret_cast<int32_t*>(ws + src_stride);  // [src_stride] codes
  __shared__ float red[4 * D];
  __shared__ float wred[NT / 32];
  __shared__ float bc[2];
  const int hq = blockIdx.x, b = blockIdx.y, h = hq / G;
  const int row = b * Hkv + h;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = merge_n[row];
  const int32_t* src = merge_src + (size_t)row * src_stride;
  const size_t hb = (size_t)b * Hq + hq;

  // pass 1: block max of the listed m
  float mx = -CUDART_INF_F;
  for (int e = tid; e < n; e += NT) {
    const int code = src[e];
    cs[e] = code;
    const float me = code < split ? m_spec[hb * w_spec + code] : m_rep[hb * w_rep + (code - split)];
    ws[e] = me;
    mx = fmaxf(mx, me);
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, off));
  if (lane == 0) wred[warp] = mx;
  __syncthreads();
  if (tid == 0) {
    float t = wred[0];
    for (int w = 1; w < NT / 32; ++w) t = fmaxf(t, wred[w]);
    bc[0] = t;
  }
  __syncthreads();
  const float m_all = bc[0];
  // pass 2: weights e^{m_e - m_all} and the denominator (fixed reduction shape -> deterministic)
  float lsum = 0.f;
  for (int e = tid; e < n; e += NT) {
    const int code = cs[e];
    const float me = ws[e];
    const float w = me == -CUDART_INF_F ? 0.f : ex2((me - m_all) * LOG2E);
    const float le = code < split ? l_spec[hb * w_spec + code] : l_rep[hb * w_rep + (code - split)];
    ws[e] = w;
    lsum = fmaf(w, le, lsum);
  }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) lsum += __shfl_xor_sync(FULL, lsum, off);
  __syncthreads();
  if (lane == 0) wred[warp] = lsum;
  __syncthreads();
  if (tid == 0) {
    float t = 0.f;
    for (int w = 0; w < NT / 32; ++w) t += wred[w];
    bc[1] = t;
  }
  __syncthreads();
  const float l_all = bc[1];
  // pass 3: O = sum_e w_e O_e ; four interleaved chains per channel, combined in a fixed order
  const int grp = tid / D, c = tid - grp * D;
  float acc = 0.f;
#pragma unroll 4
  for (int e = grp; e < n; e += 4) {
    const int code = cs[e];
    const float* Op = code < split ? O_spec + (hb * w_spec + code) * D : O_rep + (hb * w_rep + (code - split)) * D;
    acc = fmaf(ws[e], Op[c], acc);
  }
  red[tid] = acc;
  __syncthreads();
  if (grp == 0) {
    const float t = (red[c] + red[D + c]) + (red[2 * D + c] + red[3 * D + c]);
    out[hb * D + c] = l_all > 0.f ? t / l_all : 0.f;
    if (c == 0) {
      if (m_out) m_out[hb] = m_all;
      if (l_out) l_out[hb] = l_all;
    }
  }
}

// ---------------------------------------------------------------------------------------------
template <int D, int BS>
static void launch_partial_t(prr_ctx* c, const prr_paged_kv* kv, const void* q, const int32_t* list,
                             int width, float* O, float* m, float* l, cudaStream_t s) {
  dim3 grid(width, c->Hkv, kv->batch);
  if (c->lay.kv_dtype == PRR_FP8_E4M3) {
    const size_t smem = (size_t)2 * BS * (D + 8) * 2;
    if (smem > 48 * 1024)
      cudaFuncSetAttribute((const void*)k_partial<D, BS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k_partial<D, BS, true><<<grid, 2 * BS, smem, s>>>(
        (const uint16_t*)kv->k_pages, (const uint16_t*)kv->v_pages, kv->block_table, kv->seq_lens,
        (const uint16_t*)q, list, width, O, m, l, c->Hq, c->Hkv, c->G, c->MB, c->sm_scale,
        c->kscale[kv->layer], c->vscale[kv->layer]);
    return;
  }
  const size_t smem = (size_t)2 * BS * (D + 8) * 2;
  if (smem > 48 * 1024)  // (per device and cheap: not cached in a process-wide flag)
    cudaFuncSetAttribute((const void*)k_partial<D, BS, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_partial<D, BS, false><<<grid, 2 * BS, smem, s>>>(
      (const uint16_t*)kv->k_pages, (const uint16_t*)kv->v_pages, kv->block_table, kv->seq_lens,
      (const uint16_t*)q, list, width, O, m, l, c->Hq, c->Hkv, c->G, c->MB, c->sm_scale, nullptr, nullptr);
}

void launch_partial(prr_ctx* c, const prr_paged_kv* kv, const void* q, const int32_t* list,
                    int width, float* O, float* m, float* l, cudaStream_t s) {
  if (width <= 0) return;
#define PRR_CASE(DD, BB) \
  if (c->D == DD && c->bs == BB) { launch_partial_t<DD, BB>(c, kv, q, list, width, O, m, l, s); c->launches++; return; }
  PRR_CASE(128, 64) PRR_CASE(128, 32) PRR_CASE(128, 16) PRR_CASE(128, 128)
  PRR_CASE(64, 64) PRR_CASE(64, 32) PRR_CASE(64, 16) PRR_CASE(64, 128)
#undef PRR_CASE
}

void launch_merge(prr_ctx* c, int batch, const int32_t* merge_src, const int32_t* merge_n,
                  const float* O_spec, const float* m_spec, const float* l_spec, int w_spec,
                  const float* O_rep, const float* m_rep, const float* l_rep, int w_rep,
                  float* out, float* m_out, float* l_out, cudaStream_t s) {
  const int stride = c->Bud + c->K;
  const size_t smem = (size_t)stride * 8;
  dim3 grid(c->Hq, batch);
  if (c->D == 128)
    k_merge<128><<<grid, 512, smem, s>>>(merge_src, merge_n, stride, O_spec, m_spec, l_spec, w_spec,
                                         O_rep, m_rep, l_rep, w_rep, c->Bud, out, m_out, l_out,
                                         c->Hq, c->Hkv, c->G);
  else
    k_merge<64><<<grid, 256, smem, s>>>(merge_src, merge_n, stride, O_spec, m_spec, l_spec, w_spec,
                                        O_rep, m_rep, l_rep, w_rep, c->Bud, out, m_out, l_out,
                                        c->Hq, c->Hkv, c->G);
  c->launches++;
}

}  // namespace prr
