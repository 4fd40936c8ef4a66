// Host-side internals of libprr: the context and the kernel launchers (one per .cu file).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <array>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/prr.h"

struct prr_ctx {
  prr_layout lay;
  int bs, K, Bud, G, D, Hq, Hkv, MB, NL, maxB;
  float sm_scale;
  double score_c;  // 1 / (G sqrt(d)), computed once on the host in fp64

  // ---- per-layer state, device ----
  double* ema_l = nullptr;    // [NL, maxB, Hkv, MB]
  double* ema_v = nullptr;    // [NL, maxB, Hkv, MB]
  int32_t* n_state = nullptr; // [NL, maxB, Hkv]
  double* theta = nullptr;    // [NL, maxB, 3]
  double* open_sum = nullptr; // [NL, maxB, Hkv, D] running fp64 sum of the open block's keys
  float* scores = nullptr;    // [NL, maxB, Hkv, MB]
  int32_t* setA = nullptr;    // [NL, maxB, Hkv, K]
  int32_t* setM = nullptr;    // [NL, maxB, Hkv, K]
  int32_t* P_next = nullptr;  // [NL, maxB, Hkv, Bud]  prediction for the next step of the layer
  int32_t* P_used = nullptr;  // [NL, maxB, Hkv, Bud]  prediction the last step used
  // fused orchestration: the step reads Pbuf[parity[layer]] and writes the next prediction into
  // the other buffer, then flips the parity (all on the device, so a captured graph replays)
  int32_t* Pbuf[2] = {nullptr, nullptr};  // [NL, maxB, Hkv, Bud] each
  int32_t* parity = nullptr;              // [NL]
  int32_t* counts = nullptr;  // [NL, maxB, Hkv, 3]    |A|, |P|, |M| of the last step
  // ---- per-step scratch, device (shared by all layers; steps are ordered on the main stream) ----
  int32_t* merge_src = nullptr; // [maxB, Hkv, Bud+K] slot codes, ascending block order
  int32_t* merge_n = nullptr;   // [maxB, Hkv]
  int32_t* nblk = nullptr;      // [maxB] scratch for n_blocks derived from seq_lens
  float *O_spec = nullptr, *m_spec = nullptr, *l_spec = nullptr; // [maxB, Hq, Bud, D] / [.., Bud]
  float *O_rep = nullptr, *m_rep = nullptr, *l_rep = nullptr;    // [maxB, Hq, K, D]   / [.., K]
  unsigned long long* stats = nullptr; // [4]
  uint32_t* maskA = nullptr;  // [maxB, Hkv, ceil(MB/32)] bitmask of A (fused step)
  unsigned long long *mt_spec = nullptr, *mt_rep = nullptr; // [maxB, Hq, Bud+1] / [maxB, Hq, K] epoch-tagged block maxima (fused step)
  unsigned long long* ms64 = nullptr; // [maxB, Hkv, Bud+K] epoch-tagged merge lists of the running step (fused step)
  unsigned long long* sc64 = nullptr; // [maxB, Hkv, MB] epoch-tagged scores of the running step (fused step)
  unsigned long long* mtag = nullptr; // [maxB, Hkv, K] epoch-tagged missed blocks of the running step (fused step)
  float* pred = nullptr;      // [maxB, Hkv, MB] Eq. 2 predictions of the row being ranked (fused step)
  uint32_t* ctl = nullptr;    // fused step: exit counter, error flag, tickets, per-row dependency counters
  unsigned long long* tl = nullptr; int tl_on = 0, tl_warps = 0; // fused step: per-warp phase stamps (debug)
  int n_sm = 0, smem_optin = 0, fused = 1, coop = 0;
  // fused step (k_row.cu): per kernel instantiation, attribute set + co-resident clusters of 1, 2, 4, 8 CTAs
  int row_attr[6] = {0, 0, 0, 0, 0, 0}; int row_maxcl[6][5] = {}; int row_dyn[6] = {};
  int force_cs = 0, pdl = 1, cut = 1, sub_tile = 64;
  int mode = 0;                                  // PRR_MODE_S3 (EMA + repair) | _S2 (reuse + repair) | _S1 (reuse + recompute on any miss)
  int kernel = 0;                                // fused step: 0 auto, 1 persistent cooperative grid (k_step.cu), 2 cluster per row (k_row.cu)
  int summary_kind = 0;  // PRR_SUMMARY_MEAN | PRR_SUMMARY_QUEST (prr_set_option)
  int last_kernel = 0; int pace_pct = 100; float hbm_gbs_est = 6400.f; bool coop_attr[8] = {};          // tuning: cluster size override, programmatic dependent launch, early cut
  int last_cs = 0, last_nbuf = 0, last_grid = 0; // launch shape of the last fused step (introspection)
  std::unordered_map<const void*, std::array<uint64_t, 16>> tmaps; // encoded CUtensorMap per K/V page pool
  // ---- calibration scratch (allocated on first prr_calibrate) ----
  double* cal_state = nullptr; size_t cal_state_elems = 0; // [80, Hkv, N, 2]
  uint32_t* cal_mask = nullptr; size_t cal_mask_words = 0; // [Hkv, T, ceil(N/32)]
  double* cal_den = nullptr; size_t cal_den_elems = 0;     // [Hkv, T]
  double* cal_acc = nullptr;  // [80, Hkv] + counts [80, Hkv] + H [80] + best[1]
  // ---- host staging for prr_decode_step_host ----
  void *st_q = nullptr, *st_k = nullptr, *st_v = nullptr; float* st_out = nullptr;
  float* st_out_h = nullptr; float* st_out_hd = nullptr;  // small results: the kernel stores them into mapped host memory (no D2H copy)
  const void* out_seen = nullptr; float* out_seen_d = nullptr;  // last caller buffer and its device alias (null: not mapped)
  // completion word in mapped host memory: a fused step armed with arm_seq != 0 stores that value there (system-scope
  // release after its last result) so that prr_decode_step_host can poll it instead of synchronising the stream
  volatile uint32_t* done_h = nullptr; uint32_t* done_d = nullptr; uint32_t done_seq = 0, arm_seq = 0;
  void* st_pin = nullptr;  // pinned host image of [q | k_new | v_new] for one copy across PCIe

  cudaStream_t side_spec = nullptr, side_ema = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_spec = nullptr, ev_sel = nullptr;
  std::vector<cudaEvent_t> ev_upd; // per layer: EMA update of the last step of that layer done
  std::vector<char> upd_pending;
  int32_t* bud_seq = nullptr;      // [NL, maxB] device: per-sequence budget + 1, 0 = follow the layer's (prr_set_budget_seq)
  std::vector<int> bud_seq_h;      // host mirror of bud_seq
  std::vector<int> bud_eff;        // per layer: blocks predicted for the next step, 0 .. Bud (prr_set_budget)
  std::vector<double> bud_poly;    // fitted budget(context length): coefficients in x = ctx_len / bud_xscale (prr_budget_fit)
  double bud_xscale = 1.0;
  std::vector<const float*> kscale, vscale;  // per layer: fp8 scales [n_pages, Hkv] (prr_set_kv_scales), caller-owned
  std::vector<void*> allocs;
  int64_t launches = 0;
  std::string err;
};

struct prr_graph {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
};

namespace prr {

// k_cache.cu
void launch_build_summaries(prr_ctx* c, const prr_paged_kv* kv, void* summaries, cudaStream_t s);
void launch_append(prr_ctx* c, const prr_paged_kv* kv, const void* k_new, const void* v_new,
                   void* summaries, cudaStream_t s);
void launch_nblocks(prr_ctx* c, const int32_t* seq_lens, int batch, int32_t* nblk, cudaStream_t s);
// k_fp8.cu (PRR_FP8_E4M3)
void launch_quantize_fp8(prr_ctx* c, const prr_paged_kv* kv, void* k8, void* v8, float* kscale, float* vscale, cudaStream_t s);
void launch_build_summaries_fp8(prr_ctx* c, const prr_paged_kv* kv, void* summaries, cudaStream_t s);
// k_score.cu
void launch_score(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries,
                  float* scores, cudaStream_t s);
// k_select.cu
// Top-k of each row (+ optional diff against P and merge list).  n per row comes from
// seq_lens (if non-null: ceil(len/bs)) else n_blocks.
struct SelectArgs {
  const float* scores; int row_stride;
  const int32_t* seq_lens; const int32_t* n_blocks; int bs;
  int batch, Hkv, k;
  int32_t* A_out; int32_t* A_count;      // [rows,k], [rows] (count may be null)
  const int32_t* P; int Bud;             // null -> empty prediction
  int32_t* M_out;                        // [rows,k] or null
  int32_t* merge_src; int32_t* merge_n;  // [rows,Bud+k], [rows] or null
  int32_t* counts;                       // [rows,3] or null
  unsigned long long* stats;             // [4] or null
  int retain;
};
void launch_select(prr_ctx* c, const SelectArgs& a, cudaStream_t s);
// EMA update (optional) + prediction of the next P.
struct EmaArgs {
  int layer, batch, seq0;                // rows cover sequences [seq0, seq0+batch)
  const float* scores;                   // null -> predict only from the current state
  const int32_t* seq_lens; const int32_t* n_blocks; // n per sequence when updating
  int32_t* P_out; int32_t* P_count;      // [batch,Hkv,Bud], [batch,Hkv] or null
  int32_t* P_save;                       // old contents of P_out copied here first, or null
};
void launch_ema(prr_ctx* c, const EmaArgs& a, cudaStream_t s);
// k_attn.cu
void launch_partial(prr_ctx* c, const prr_paged_kv* kv, const void* q, const int32_t* list,
                    int width, float* O, float* m, float* l, cudaStream_t s);
void launch_merge(prr_ctx* c, int batch, const int32_t* merge_src, const int32_t* merge_n,
                  const float* O_spec, const float* m_spec, const float* l_spec, int w_spec,
                  const float* O_rep, const float* m_rep, const float* l_rep, int w_rep,
                  float* out, float* m_out, float* l_out, cudaStream_t s);
// One fused launch for a whole layer-step; spec = 0 is the sequential path.  Returns 0 or a cudaError_t.
// k_step.cu: one persistent cooperative grid, warps as workers, global-memory flags between the stages
// (best when the rows are few: batch 1).  k_row.cu: one thread-block cluster per (sequence, KV head) row,
// everything between the stages of a row on chip (best when the rows fill the GPU).
int launch_step_persist(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries, float* out,
                        int spec, cudaStream_t s, const void* k_new, const void* v_new);
int launch_step_cluster(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries, float* out,
                        int spec, cudaStream_t s, const void* k_new, const void* v_new);
// k_calib.cu
int launch_calibrate(prr_ctx* c, int layer, int seq, const float* IS, int T, int N,
                     const int32_t* n_valid, cudaStream_t s);

}  // namespace prr
