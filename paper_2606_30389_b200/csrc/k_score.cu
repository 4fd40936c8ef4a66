// a1 — block-importance scoring ("compressed attention", group aggregation as in A.1
// PAPER.md:372): IS[b,h,i] = fp32( (sum_g sum_j q[b,hG+g,j] kbar[b,h,i,j]) / (G sqrt d) ).
//
// HBM-bound stream over the summary rows (d bf16 each).  A sub-warp of d/8 lanes owns one row with
// one 16-byte load per lane; the group's queries are pre-summed per channel in fp64 (exact), the
// 8 products per lane are exact fp64 FMAs, and the sub-warp is reduced with shuffles.  Because
// every intermediate is exactly representable (bf16 x small-integer-sum products, Q1)
// the sum is order-independent and the single RNE to fp32 matches the oracle bit for bit.
//
// QUEST = true scores Quest's channel-wise min / max metadata with the same GQA mean query (A.1,
// PAPER.md:372): IS[b,h,i] = fp32( (sum_j max(qs_j m[b,h,i,j], qs_j M[b,h,i,j])) / (G sqrt d) ); a row is
// then 2 d bf16 (min then max), each lane loads both halves of its 8 channels; every term is one of
// two exact products, so the sum stays order-independent.
#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {

template <int D, bool QUEST>
__global__ void __launch_bounds__(256)
k_score(const uint4* __restrict__ summ, const uint16_t* __restrict__ q,
        const int32_t* __restrict__ seq_lens, float* __restrict__ scores, int Hq, int Hkv, int G,
        int MB, int bs, double c) {
  constexpr int LPR = D / 8;        // lanes per row
  constexpr int RW = 32 / LPR;      // rows per warp per iteration
  constexpr int UNR = QUEST ? 2 : 4;  // independent rows in flight per lane (one or two 16-B loads each)
  constexpr int RS = QUEST ? 2 * LPR : LPR;  // row stride in uint4
  constexpr int ROWS_CTA = 8 * RW * UNR;
  const int b = blockIdx.z, h = blockIdx.y;
  const int nb = min(MB, (seq_lens[b] + bs - 1) / bs);
  const int row0 = blockIdx.x * ROWS_CTA;
  if (row0 >= nb) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sub = lane / LPR, l = lane % LPR;

  const uint4* rows = summ + ((size_t)b * Hkv + h) * MB * RS;
  const int rbase = row0 + warp * RW * UNR + sub;
  uint4 v[UNR], vM[UNR];
#pragma unroll
  for (int u = 0; u < UNR; ++u) {
    const int r = rbase + u * RW;
    v[u] = r < nb ? __ldg(rows + (size_t)r * RS + l) : make_uint4(0, 0, 0, 0);
    vM[u] = QUEST && r < nb ? __ldg(rows + (size_t)r * RS + LPR + l) : make_uint4(0, 0, 0, 0);
  }

  double qs[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) qs[j] = 0.0;
  const uint16_t* qb = q + ((size_t)b * Hq + (size_t)h * G) * D + l * 8;
  for (int g = 0; g < G; ++g) {
    const uint4 t = __ldg(reinterpret_cast<const uint4*>(qb + (size_t)g * D));
    const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      qs[2 * j] += (double)bf16_lo(w[j]);
      qs[2 * j + 1] += (double)bf16_hi(w[j]);
    }
  }

#pragma unroll
  for (int u = 0; u < UNR; ++u) {
    const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
    double acc = 0.0;
    if (QUEST) {
      const uint32_t wM[4] = {vM[u].x, vM[u].y, vM[u].z, vM[u].w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        acc += fmax(__dmul_rn((double)bf16_lo(w[j]), qs[2 * j]), __dmul_rn((double)bf16_lo(wM[j]), qs[2 * j]));
        acc += fmax(__dmul_rn((double)bf16_hi(w[j]), qs[2 * j + 1]), __dmul_rn((double)bf16_hi(wM[j]), qs[2 * j + 1]));
      }
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        acc = fma((double)bf16_lo(w[j]), qs[2 * j], acc);
        acc = fma((double)bf16_hi(w[j]), qs[2 * j + 1], acc);
      }
    }
#pragma unroll
    for (int off = LPR / 2; off >= 1; off >>= 1) acc += __shfl_xor_sync(FULL, acc, off);
    const int r = rbase + u * RW;
    if (l == 0 && r < nb) scores[((size_t)b * Hkv + h) * MB + r] = f64_to_score(__dmul_rn(acc, c));
  }
}

void launch_score(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries,
                  float* scores, cudaStream_t s) {
  const bool quest = c->summary_kind == PRR_SUMMARY_QUEST;
  const int rows_cta = (c->D == 128 ? 64 : 128) / (quest ? 2 : 1);
  dim3 grid((c->MB + rows_cta - 1) / rows_cta, c->Hkv, kv->batch);
#define PRR_SCORE(DD, QQ)                                                                              \
  k_score<DD, QQ><<<grid, 256, 0, s>>>((const uint4*)summaries, (const uint16_t*)q, kv->seq_lens, scores, \
                                       c->Hq, c->Hkv, c->G, c->MB, c->bs, c->score_c)
  if (c->D == 128) { if (quest) PRR_SCORE(128, true); else PRR_SCORE(128, false); }
  else { if (quest) PRR_SCORE(64, true); else PRR_SCORE(64, false); }
#undef PRR_SCORE
  c->launches++;
}

}  // namespace prr
