// a2 top-K (+ a5 diff) and a3/a8 the EMA predictor.
//
// k_select: one CTA per (sequence, KV head) row.  Radix select on order-preserving uint32 keys of
// the fp32 scores held in shared memory (A.1 PAPER.md:372: K highest-scoring
// blocks per KV head, shared by the group; ties -> lower block index), ordered compaction to an
// ascending list + bitmask, then the diff against the predicted set P (PAPER.md:102-105:
// M = A\P, N = P\A) emitted as the slot list the merge kernel folds in ascending block order.
//
// k_ema: one CTA per row.  Eq. 3 update (first-seen blocks l = IS, v = 0,
// PAPER.md:137) in non-contracted fp64, Eq. 2 prediction rounded once to fp32, and
// the same radix select for P = top-min(Bud, #stateful) (Eq. 1).
#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {

constexpr int SEL_NT = 256;

struct SelSmem {
  unsigned long long* scan;  // 40 x u64
  uint32_t* keys;            // [row_stride]
  uint32_t* maskA;           // [words]
  uint32_t* maskP;           // [words]
  uint32_t* hist;            // [256]
  uint32_t* ctl;             // [8]
};
__device__ __forceinline__ SelSmem carve(unsigned char* base, int row_stride, int words) {
  SelSmem s;
  s.scan = reinterpret_cast<unsigned long long*>(base);
  s.keys = reinterpret_cast<uint32_t*>(base + 40 * 8);
  s.maskA = s.keys + row_stride;
  s.maskP = s.maskA + words;
  s.hist = s.maskP + words;
  s.ctl = s.hist + 256;
  return s;
}
static size_t sel_smem_bytes(int row_stride) {
  const int words = (row_stride + 31) / 32;
  return 40 * 8 + ((size_t)row_stride + 2 * words + 256 + 8) * 4;
}

__global__ void __launch_bounds__(SEL_NT) k_select(SelectArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x;
  const int row = blockIdx.x, b = row / a.Hkv;
  const int words = (a.row_stride + 31) / 32;
  SelSmem s = carve(smem_raw, a.row_stride, words);
  int n = a.seq_lens ? (a.seq_lens[b] + a.bs - 1) / a.bs : a.n_blocks[b];
  n = max(0, min(n, a.row_stride));

  for (int w = tid; w < 2 * words; w += SEL_NT) s.maskA[w] = 0;  // maskA and maskP are adjacent
  int32_t* A_row = a.A_out + (size_t)row * a.k;
  if (a.scores) {
    const float* sc = a.scores + (size_t)row * a.row_stride;
    for (int i = tid; i < n; i += SEL_NT) s.keys[i] = score_key(sc[i]);
    __syncthreads();
    const int k = min(a.k, n);
    int cntA = 0;
    if (k > 0) {
      uint32_t T;
      int need;
      radix_select<SEL_NT>(s.keys, n, k, s.hist, s.ctl, T, need);
      cntA = ordered_select<SEL_NT>(s.keys, n, T, need, A_row, s.maskA, s.scan);
    }
    for (int j = cntA + tid; j < a.k; j += SEL_NT) A_row[j] = -1;
    if (a.A_count && tid == 0) a.A_count[row] = cntA;
  } else {  // A is given (prr_repair): build its bitmask from the list
    __syncthreads();
    for (int j = tid; j < a.k; j += SEL_NT) {
      const int blk = A_row[j];
      if (blk >= 0 && blk < a.row_stride) atomicOr(&s.maskA[blk >> 5], 1u << (blk & 31));
    }
  }
  if (!a.merge_src && !a.M_out && !a.counts && !a.stats) return;

  if (a.P) {
    const int32_t* P_row = a.P + (size_t)row * a.Bud;
    for (int j = tid; j < a.Bud; j += SEL_NT) {
      const int blk = P_row[j];
      if (blk >= 0 && blk < a.row_stride) atomicOr(&s.maskP[blk >> 5], 1u << (blk & 31));
    }
  }
  __syncthreads();

  // Walk the bit words in ascending block order.  Packed counters, 16 bits each (<= 32768):
  // U (blocks to merge) | P | M = A\P | A.
  const int wper = (words + SEL_NT - 1) / SEL_NT;
  const int w0 = min(words, tid * wper), w1 = min(words, w0 + wper);
  unsigned long long loc = 0;
  for (int w = w0; w < w1; ++w) {
    const uint32_t A = s.maskA[w], P = s.maskP[w];
    const uint32_t U = a.retain ? (A | P) : A;
    loc += ((unsigned long long)__popc(U) << 48) | ((unsigned long long)__popc(P) << 32) |
           ((unsigned long long)__popc(A & ~P) << 16) | (unsigned long long)__popc(A);
  }
  unsigned long long tot;
  const unsigned long long ex = block_excl_scan<SEL_NT>(loc, s.scan, &tot);
  int upos = (int)(ex >> 48), prank = (int)((ex >> 32) & 0xffffu), mrank = (int)((ex >> 16) & 0xffffu);
  const int nU = (int)(tot >> 48), nP = (int)((tot >> 32) & 0xffffu),
            nM = (int)((tot >> 16) & 0xffffu), nA = (int)(tot & 0xffffu);
  int32_t* src_row = a.merge_src ? a.merge_src + (size_t)row * (a.Bud + a.k) : nullptr;
  int32_t* M_row = a.M_out ? a.M_out + (size_t)row * a.k : nullptr;
  for (int w = w0; w < w1; ++w) {
    const uint32_t A = s.maskA[w], P = s.maskP[w];
    uint32_t U = a.retain ? (A | P) : A;
    const uint32_t Mw = A & ~P;
    while (U) {
      const int bit = __ffs(U) - 1;
      U &= U - 1;
      const uint32_t below = (1u << bit) - 1u;
      int code;
      if ((P >> bit) & 1u) {
        code = prank + __popc(P & below);          // slot in the speculative partials
      } else {
        const int j = mrank + __popc(Mw & below);  // slot in the repair partials
        code = a.Bud + j;
        if (M_row) M_row[j] = w * 32 + bit;
      }
      if (src_row) src_row[upos] = code;
      ++upos;
    }
    prank += __popc(P);
    mrank += __popc(Mw);
  }
  if (M_row)
    for (int j = nM + tid; j < a.k; j += SEL_NT) M_row[j] = -1;
  if (tid == 0) {
    if (a.merge_n) a.merge_n[row] = nU;
    if (a.counts) {
      a.counts[row * 3 + 0] = nA;
      a.counts[row * 3 + 1] = nP;
      a.counts[row * 3 + 2] = nM;
    }
    if (a.stats) {
      atomicAdd(&a.stats[0], (unsigned long long)nA);
      atomicAdd(&a.stats[1], (unsigned long long)(nA - nM));
      atomicAdd(&a.stats[2], (unsigned long long)nM);
      atomicAdd(&a.stats[3], (unsigned long long)nP);
    }
  }
}

// ---------------------------------------------------------------------------------------------
struct EmaKArgs {
  double* ema_l; double* ema_v; int32_t* n_state; const double* theta;  // already offset to (layer, seq0)
  const float* scores; const int32_t* seq_lens; const int32_t* n_blocks;
  int32_t* P_out; int32_t* P_count; int32_t* P_save;
  int Hkv, MB, Bud, BudSel, bs;  // Bud: width of a P row; BudSel <= Bud: blocks predicted (the run-time budget)
  const int32_t* bud_seq;        // per sequence (already offset): 0 = the layer's budget, v > 0 = budget v - 1
};

__global__ void __launch_bounds__(SEL_NT) k_ema(EmaKArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x;
  const int row = blockIdx.x, bi = row / a.Hkv;
  const int words = (a.MB + 31) / 32;
  SelSmem s = carve(smem_raw, a.MB, words);
  double* L = a.ema_l + (size_t)row * a.MB;
  double* V = a.ema_v + (size_t)row * a.MB;
  const double alpha = a.theta[bi * 3 + 0], beta = a.theta[bi * 3 + 1], gamma = a.theta[bi * 3 + 2];
  const int n_old = a.n_state[row];
  int n_new = n_old;
  if (a.scores) {
    int n = a.seq_lens ? (a.seq_lens[bi] + a.bs - 1) / a.bs : a.n_blocks[bi];
    n = max(0, min(n, a.MB));
    n_new = max(n, n_old);
    const double oma = __dsub_rn(1.0, alpha), omb = __dsub_rn(1.0, beta);
    const float* sc = a.scores + (size_t)row * a.MB;
    for (int i = tid; i < n_new; i += SEL_NT) {
      double ln, vn;
      if (i < n) {
        const double x = (double)sc[i];
        if (i < n_old) {  // Eq. 3, both lines use l^{t-1}; one IEEE operation per parenthesis
          const double lo = L[i], vo = V[i];
          vn = __dadd_rn(__dmul_rn(beta, __dsub_rn(x, lo)), __dmul_rn(omb, vo));
          ln = __dadd_rn(__dmul_rn(alpha, x), __dmul_rn(oma, lo));
        } else {          // first time this block is scored
          ln = x;
          vn = 0.0;
        }
        L[i] = ln;
        V[i] = vn;
      } else {
        ln = L[i];
        vn = V[i];
      }
      s.keys[i] = score_key(f64_to_score(__dadd_rn(ln, __dmul_rn(gamma, vn))));
    }
  } else {
    for (int i = tid; i < n_old; i += SEL_NT)
      s.keys[i] = score_key(f64_to_score(__dadd_rn(L[i], __dmul_rn(gamma, V[i]))));
  }
  int32_t* P_row = a.P_out + (size_t)row * a.Bud;
  if (a.P_save)
    for (int j = tid; j < a.Bud; j += SEL_NT) a.P_save[(size_t)row * a.Bud + j] = P_row[j];
  __syncthreads();
  if (a.scores && tid == 0) a.n_state[row] = n_new;
  const int bsel = a.bud_seq[bi] > 0 ? min(a.bud_seq[bi] - 1, a.Bud) : a.BudSel;  // (prr_set_budget_seq)
  const int k = min(bsel, n_new);
  int cnt = 0;
  if (k > 0) {
    uint32_t T;
    int need;
    radix_select<SEL_NT>(s.keys, n_new, k, s.hist, s.ctl, T, need);
    cnt = ordered_select<SEL_NT>(s.keys, n_new, T, need, P_row, nullptr, s.scan);
  }
  for (int j = cnt + tid; j < a.Bud; j += SEL_NT) P_row[j] = -1;
  if (a.P_count && tid == 0) a.P_count[row] = cnt;
}

// ---------------------------------------------------------------------------------------------
static void ensure_smem(const void* fn, size_t bytes) {
  if (bytes > 48 * 1024)
    cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

void launch_select(prr_ctx* c, const SelectArgs& a, cudaStream_t s) {
  const size_t smem = sel_smem_bytes(a.row_stride);
  ensure_smem((const void*)k_select, smem);
  k_select<<<a.batch * a.Hkv, SEL_NT, smem, s>>>(a);
  c->launches++;
}

void launch_ema(prr_ctx* c, const EmaArgs& e, cudaStream_t s) {
  if (c->Bud <= 0 && !e.scores) return;
  EmaKArgs a;
  const size_t seq = (size_t)e.layer * c->maxB + e.seq0;
  a.ema_l = c->ema_l + seq * c->Hkv * c->MB;
  a.ema_v = c->ema_v + seq * c->Hkv * c->MB;
  a.n_state = c->n_state + seq * c->Hkv;
  a.theta = c->theta + seq * 3;
  a.scores = e.scores;
  a.seq_lens = e.seq_lens;
  a.n_blocks = e.n_blocks;
  a.P_out = e.P_out;
  a.P_count = e.P_count;
  a.P_save = e.P_save;
  a.Hkv = c->Hkv;
  a.MB = c->MB;
  a.Bud = c->Bud;
  a.BudSel = c->bud_eff[e.layer];
  a.bud_seq = c->bud_seq + (size_t)e.layer * c->maxB + e.seq0;
  a.bs = c->bs;
  const size_t smem = sel_smem_bytes(c->MB);
  ensure_smem((const void*)k_ema, smem);
  k_ema<<<e.batch * c->Hkv, SEL_NT, smem, s>>>(a);
  c->launches++;
}

}  // namespace prr
