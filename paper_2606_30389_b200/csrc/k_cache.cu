// a0 — paged-cache maintenance: bulk mean-key summaries, single-token append with summary refresh.
// PAPER.md:66 "partitions KV tokens into blocks, compresses each block (e.g., mean)".
#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {

// One CTA per (block, KV head, sequence); thread c owns channel c.  Sum of <= 128 bf16 values in
// fp64 is exact, so the mean is one correctly rounded division followed by one RNE to bf16 (Q2).
__global__ void k_build_summaries(const uint16_t* __restrict__ kp, const int32_t* __restrict__ table,
                                  const int32_t* __restrict__ seq_lens, uint16_t* __restrict__ summ,
                                  double* __restrict__ open_sum, int Hkv, int bs, int D, int MB) {
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z, c = threadIdx.x;
  const int len = seq_lens[b];
  const int nb = (len + bs - 1) / bs;
  if (i >= nb) return;
  const int n_i = min(bs, len - i * bs);
  const size_t page = (size_t)table[(size_t)b * MB + i];
  const uint16_t* src = kp + ((page * Hkv + h) * bs) * (size_t)D + c;
  double s = 0.0;
  for (int t = 0; t < n_i; ++t) s += bf16_to_f64(src[(size_t)t * D]);
  summ[(((size_t)b * Hkv + h) * MB + i) * D + c] = f64_to_bf16_rne(__ddiv_rn(s, (double)n_i));
  if (i == nb - 1) open_sum[((size_t)b * Hkv + h) * D + c] = s;
}

// Quest's page metadata (A.1): channel-wise minimum and maximum key of the block's valid tokens,
// row layout [2][D] (min then max).  A min / max of bf16 values is one of them: no rounding anywhere.
__global__ void k_build_minmax(const uint16_t* __restrict__ kp, const int32_t* __restrict__ table,
                               const int32_t* __restrict__ seq_lens, uint16_t* __restrict__ summ, int Hkv, int bs,
                               int D, int MB) {
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z, c = threadIdx.x;
  const int len = seq_lens[b];
  const int nb = (len + bs - 1) / bs;
  if (i >= nb) return;
  const int n_i = min(bs, len - i * bs);
  const size_t page = (size_t)table[(size_t)b * MB + i];
  const uint16_t* src = kp + ((page * Hkv + h) * bs) * (size_t)D + c;
  uint16_t lo = src[0], hi = lo;
  for (int t = 1; t < n_i; ++t) {
    const uint16_t x = src[(size_t)t * D];
    if (bf16_to_f64(x) < bf16_to_f64(lo)) lo = x;
    if (bf16_to_f64(x) > bf16_to_f64(hi)) hi = x;
  }
  uint16_t* dst = summ + (((size_t)b * Hkv + h) * MB + i) * 2 * D;
  dst[c] = lo;
  dst[D + c] = hi;
}

// One CTA per sequence.  Token position = seq_lens[b] (before the append).
__global__ void k_append(uint16_t* __restrict__ kp, uint16_t* __restrict__ vp,
                         const int32_t* __restrict__ table, int32_t* __restrict__ seq_lens,
                         const uint16_t* __restrict__ k_new, const uint16_t* __restrict__ v_new,
                         uint16_t* __restrict__ summ, double* __restrict__ open_sum, int Hkv, int bs,
                         int D, int MB, int quest) {
  const int b = blockIdx.x;
  const int pos = seq_lens[b];
  const int blk = pos / bs, slot = pos - blk * bs;
  if (blk >= MB) return;  // the sequence is full: nothing is written, the length stays (the caller maps max_blocks_per_seq pages)
  const size_t page = (size_t)table[(size_t)b * MB + blk];
  for (int idx = threadIdx.x; idx < Hkv * D; idx += blockDim.x) {
    const int h = idx / D, c = idx - h * D;
    const uint16_t kk = k_new[(size_t)b * Hkv * D + idx];
    const size_t dst = ((page * Hkv + h) * bs + slot) * (size_t)D + c;
    kp[dst] = kk;
    vp[dst] = v_new[(size_t)b * Hkv * D + idx];
    if (quest) {  // the open block's min / max absorb the token; a block's first token starts both
      uint16_t* mm = summ + (((size_t)b * Hkv + h) * MB + blk) * 2 * D;
      if (slot == 0 || bf16_to_f64(kk) < bf16_to_f64(mm[c])) mm[c] = kk;
      if (slot == 0 || bf16_to_f64(kk) > bf16_to_f64(mm[D + c])) mm[D + c] = kk;
      continue;
    }
    const size_t so = ((size_t)b * Hkv + h) * D + c;
    const double x = bf16_to_f64(kk);
    const double s = slot == 0 ? x : __dadd_rn(open_sum[so], x);
    open_sum[so] = s;
    summ[(((size_t)b * Hkv + h) * MB + blk) * D + c] =
        f64_to_bf16_rne(__ddiv_rn(s, (double)(slot + 1)));
  }
  __syncthreads();
  if (threadIdx.x == 0) seq_lens[b] = pos + 1;
}

__global__ void k_nblocks(const int32_t* __restrict__ seq_lens, int32_t* __restrict__ nblk, int batch,
                          int bs) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < batch) nblk[b] = (seq_lens[b] + bs - 1) / bs;
}

void launch_build_summaries(prr_ctx* c, const prr_paged_kv* kv, void* summaries, cudaStream_t s) {
  if (c->lay.kv_dtype == PRR_FP8_E4M3) { launch_build_summaries_fp8(c, kv, summaries, s); return; }
  dim3 grid(c->MB, c->Hkv, kv->batch);
  if (c->summary_kind == PRR_SUMMARY_QUEST) {
    k_build_minmax<<<grid, c->D, 0, s>>>((const uint16_t*)kv->k_pages, kv->block_table, kv->seq_lens,
                                         (uint16_t*)summaries, c->Hkv, c->bs, c->D, c->MB);
    c->launches++;
    return;
  }
  double* os = c->open_sum + (size_t)kv->layer * c->maxB * c->Hkv * c->D;
  k_build_summaries<<<grid, c->D, 0, s>>>((const uint16_t*)kv->k_pages, kv->block_table,
                                          kv->seq_lens, (uint16_t*)summaries, os, c->Hkv, c->bs,
                                          c->D, c->MB);
  c->launches++;
}

void launch_append(prr_ctx* c, const prr_paged_kv* kv, const void* k_new, const void* v_new,
                   void* summaries, cudaStream_t s) {
  double* os = c->open_sum + (size_t)kv->layer * c->maxB * c->Hkv * c->D;
  k_append<<<kv->batch, 256, 0, s>>>((uint16_t*)kv->k_pages, (uint16_t*)kv->v_pages,
                                     kv->block_table, kv->seq_lens, (const uint16_t*)k_new,
                                     (const uint16_t*)v_new, (uint16_t*)summaries, os, c->Hkv,
                                     c->bs, c->D, c->MB, c->summary_kind == PRR_SUMMARY_QUEST);
  c->launches++;
}

void launch_nblocks(prr_ctx* c, const int32_t* seq_lens, int batch, int32_t* nblk, cudaStream_t s) {
  k_nblocks<<<(batch + 127) / 128, 128, 0, s>>>(seq_lens, nblk, batch, c->bs);
  c->launches++;
}

}  // namespace prr
