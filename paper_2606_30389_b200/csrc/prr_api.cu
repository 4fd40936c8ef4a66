// C-ABI entry points of libprr (include/prr.h): argument validation, state allocation and the
// two-stream, event-ordered orchestration of one PRR layer-step (Fig. 1, :38-42).
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <algorithm>
#include <cstring>

#include "prr_internal.h"

static constexpr size_t HOST_OUT_DIRECT = 64 << 10;  // results up to this size are stored into host memory by the kernel


using namespace prr;

static thread_local std::string g_create_err;

#define PRR_FAIL(ctx, code, ...)                      \
  do {                                                \
    char _b[512];                                     \
    snprintf(_b, sizeof(_b), __VA_ARGS__);            \
    if (ctx) (ctx)->err = _b; else g_create_err = _b; \
    return (code);                                    \
  } while (0)

#define PRR_CUDA(ctx, expr)                                                            \
  do {                                                                                 \
    cudaError_t _e = (expr);                                                           \
    if (_e != cudaSuccess) PRR_FAIL(ctx, PRR_E_CUDA, "%s: %s", #expr, cudaGetErrorString(_e)); \
  } while (0)

static int check_launch(prr_ctx* c, const char* what) {
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) {
    cudaGetLastError();
    PRR_FAIL(c, PRR_E_CUDA, "%s: %s", what, cudaGetErrorString(e));
  }
  return PRR_OK;
}

static size_t layer_rows(const prr_ctx* c, int layer) { return (size_t)layer * c->maxB * c->Hkv; }

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <typename T>
static cudaError_t dalloc(prr_ctx* c, T** p, size_t n, bool zero = true) {
  void* q = nullptr;
  cudaError_t e = cudaMalloc(&q, n * sizeof(T) + 16);
  if (e != cudaSuccess) return e;
  c->allocs.push_back(q);
  if (zero) e = cudaMemset(q, 0, n * sizeof(T) + 16);
  *p = reinterpret_cast<T*>(q);
  return e;
}

extern "C" const char* prr_version(void) { return "prr-b200 0.1 (sm_100a)"; }

extern "C" const char* prr_last_error(const prr_ctx* ctx) {
  return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

extern "C" int64_t prr_launch_count(const prr_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int32_t prr_create(const prr_layout* lay, int32_t block_size, int32_t K, int32_t budget,
                              prr_ctx** out) {
  prr_ctx* none = nullptr;
  if (!lay || !out) PRR_FAIL(none, PRR_E_INVALID, "prr_create: null argument");
  *out = nullptr;
  if (lay->n_q_heads <= 0 || lay->n_kv_heads <= 0 || lay->n_q_heads % lay->n_kv_heads)
    PRR_FAIL(none, PRR_E_INVALID, "prr_create: n_q_heads must be a positive multiple of n_kv_heads");
  if (lay->max_batch < 1 || lay->n_layers < 1 || lay->max_blocks_per_seq < 1)
    PRR_FAIL(none, PRR_E_INVALID, "prr_create: max_batch, n_layers, max_blocks_per_seq must be >= 1");
  if (K < 1 || budget < 0) PRR_FAIL(none, PRR_E_INVALID, "prr_create: need K >= 1 and budget >= 0");
  if (lay->overpredict_policy != PRR_DROP && lay->overpredict_policy != PRR_RETAIN)
    PRR_FAIL(none, PRR_E_INVALID, "prr_create: unknown overpredict_policy");
  if (lay->orchestration != PRR_FUSED && lay->orchestration != PRR_STREAMS)
    PRR_FAIL(none, PRR_E_INVALID, "prr_create: unknown orchestration");
  if (lay->sm_scale < 0.f || lay->sm_scale != lay->sm_scale)
    PRR_FAIL(none, PRR_E_INVALID, "prr_create: sm_scale must be >= 0");
  const int G = lay->n_q_heads / lay->n_kv_heads;
  if (lay->head_dim != 64 && lay->head_dim != 128)
    PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: head_dim must be 64 or 128");
  if (block_size != 16 && block_size != 32 && block_size != 64 && block_size != 128 && block_size != 256)
    PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: block_size must be 16, 32, 64, 128 or 256");
  if (block_size == 256 && lay->orchestration != PRR_FUSED)
    PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: block_size 256 needs PRR_FUSED");
  if (G > 16) PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: GQA group > 16 unsupported");
  if (lay->kv_dtype != PRR_BF16 && lay->kv_dtype != PRR_FP8_E4M3)
    PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: kv_dtype must be PRR_BF16 or PRR_FP8_E4M3");
  if (lay->kv_dtype == PRR_FP8_E4M3 && (lay->orchestration != PRR_STREAMS || block_size > 128))
    PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: PRR_FP8_E4M3 needs PRR_STREAMS and block_size <= 128");
  if (lay->max_blocks_per_seq > 32768 || K > 512 || budget > 1024)
    PRR_FAIL(none, PRR_E_UNSUPPORTED, "prr_create: max_blocks_per_seq <= 32768, K <= 512, budget <= 1024");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    PRR_FAIL(none, PRR_E_CUDA, "prr_create: no CUDA device (this library has no CPU fallback)");
  }
  prr_ctx* c = new prr_ctx();
  c->lay = *lay;
  c->bs = block_size; c->K = K; c->Bud = budget; c->G = G; c->D = lay->head_dim;
  c->Hq = lay->n_q_heads; c->Hkv = lay->n_kv_heads; c->MB = lay->max_blocks_per_seq;
  c->NL = lay->n_layers; c->maxB = lay->max_batch;
  c->sm_scale = lay->sm_scale > 0.f ? lay->sm_scale : (float)(1.0 / std::sqrt((double)c->D));
  c->score_c = 1.0 / ((double)G * std::sqrt((double)c->D));
  c->fused = lay->orchestration == PRR_FUSED;
  {
    int dev = 0, coop = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    c->coop = coop;
    if (c->n_sm < 1) {
      delete c;
      PRR_FAIL(none, PRR_E_CUDA, "prr_create: no multiprocessors reported");
    }
    int mclk = 0, bus = 0;
    cudaDeviceGetAttribute(&mclk, cudaDevAttrMemoryClockRate, dev);     // kHz
    cudaDeviceGetAttribute(&bus, cudaDevAttrGlobalMemoryBusWidth, dev); // bits
    if (mclk > 0 && bus > 0) c->hbm_gbs_est = 0.8f * 2.0f * (float)mclk * 1e3f * (float)bus / 8.0f / 1e9f;
  }

  const size_t rows = (size_t)c->NL * c->maxB * c->Hkv;
  const size_t srows = (size_t)c->maxB * c->Hkv;
  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  A(dalloc(c, &c->ema_l, rows * c->MB));
  A(dalloc(c, &c->ema_v, rows * c->MB));
  A(dalloc(c, &c->n_state, rows));
  A(dalloc(c, &c->theta, (size_t)c->NL * c->maxB * 3));
  A(dalloc(c, &c->bud_seq, (size_t)c->NL * c->maxB));
  A(dalloc(c, &c->open_sum, rows * c->D));
  A(dalloc(c, &c->scores, rows * c->MB));
  A(dalloc(c, &c->setA, rows * c->K));
  A(dalloc(c, &c->setM, rows * c->K));
  A(dalloc(c, &c->P_next, rows * (size_t)(c->Bud + 1)));
  A(dalloc(c, &c->P_used, rows * (size_t)(c->Bud + 1)));
  A(dalloc(c, &c->counts, rows * 3));
  A(dalloc(c, &c->Pbuf[0], rows * (size_t)(c->Bud + 1)));
  A(dalloc(c, &c->Pbuf[1], rows * (size_t)(c->Bud + 1)));
  A(dalloc(c, &c->parity, (size_t)c->NL));
  A(dalloc(c, &c->maskA, srows * (size_t)((c->MB + 31) / 32)));
  A(dalloc(c, &c->pred, srows * (size_t)c->MB));
  A(dalloc(c, &c->mtag, srows * (size_t)c->K));
  A(dalloc(c, &c->sc64, srows * (size_t)c->MB));
  A(dalloc(c, &c->ms64, srows * (size_t)(c->Bud + c->K)));
  A(dalloc(c, &c->ctl, (size_t)10 + srows * ((size_t)3 + c->Bud + c->K + c->MB)));  // header + flag arrays (k_step.cu)
  c->tl_warps = c->n_sm * 32;
  {  // phase stamps live in pinned, device-mapped HOST memory: readable while a step runs or after a fault
    void* p = nullptr;
    if (e == cudaSuccess) e = cudaHostAlloc(&p, (size_t)c->tl_warps * 16 * sizeof(unsigned long long), cudaHostAllocMapped);
    if (e == cudaSuccess) { memset(p, 0, (size_t)c->tl_warps * 16 * sizeof(unsigned long long)); c->tl = (unsigned long long*)p; }
  }
  A(dalloc(c, &c->merge_src, srows * (c->Bud + c->K)));
  A(dalloc(c, &c->merge_n, srows));
  A(dalloc(c, &c->nblk, (size_t)c->maxB));
  const size_t qrows = (size_t)c->maxB * c->Hq;
  A(dalloc(c, &c->O_spec, qrows * (size_t)(c->Bud + 1) * c->D, false));
  A(dalloc(c, &c->m_spec, qrows * (size_t)(c->Bud + 1), false));
  A(dalloc(c, &c->l_spec, qrows * (size_t)(c->Bud + 1), false));
  A(dalloc(c, &c->O_rep, qrows * c->K * c->D, false));
  A(dalloc(c, &c->m_rep, qrows * c->K, false));
  A(dalloc(c, &c->l_rep, qrows * c->K, false));
  A(dalloc(c, &c->mt_spec, qrows * (size_t)(c->Bud + 1)));
  A(dalloc(c, &c->mt_rep, qrows * (size_t)c->K));
  A(dalloc(c, &c->stats, (size_t)4));
  A(dalloc(c, &c->cal_acc, (size_t)2 * 80 * c->Hkv + 80 + 2));
  // host-buffer entry point: q | k_new | v_new are staged in ONE pinned buffer and cross PCIe as ONE copy
  uint16_t* sq = nullptr;
  const size_t st_elems = (qrows + 2 * srows) * c->D;   // (every part is a multiple of 16 bytes: D >= 64)
  A(dalloc(c, &sq, st_elems));
  A(dalloc(c, &c->st_out, qrows * c->D));
  c->st_q = sq; c->st_k = sq ? sq + qrows * c->D : nullptr; c->st_v = sq ? sq + (qrows + srows) * c->D : nullptr;
  if (e == cudaSuccess) e = cudaHostAlloc(&c->st_pin, st_elems * sizeof(uint16_t), cudaHostAllocDefault);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->st_out_h, std::min(qrows * c->D * sizeof(float), (size_t)HOST_OUT_DIRECT), cudaHostAllocMapped);
  if (e == cudaSuccess) e = cudaHostGetDevicePointer((void**)&c->st_out_hd, c->st_out_h, 0);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->done_h, 64, cudaHostAllocMapped);
  if (e == cudaSuccess) { *c->done_h = 0u; e = cudaHostGetDevicePointer((void**)&c->done_d, (void*)c->done_h, 0); }
  if (e == cudaSuccess) {
    // P lists start empty (-1); theta defaults to (1, 1, 0): "reuse the last step's top-K" (S1)
    e = cudaMemset(c->P_next, 0xff, rows * (size_t)(c->Bud + 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemset(c->P_used, 0xff, rows * (size_t)(c->Bud + 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemset(c->Pbuf[0], 0xff, rows * (size_t)(c->Bud + 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemset(c->Pbuf[1], 0xff, rows * (size_t)(c->Bud + 1) * sizeof(int32_t));
    std::vector<double> th((size_t)c->NL * c->maxB * 3);
    for (size_t i = 0; i < th.size(); i += 3) { th[i] = 1.0; th[i + 1] = 1.0; th[i + 2] = 0.0; }
    if (e == cudaSuccess) e = cudaMemcpy(c->theta, th.data(), th.size() * sizeof(double), cudaMemcpyHostToDevice);
  }
  A(cudaStreamCreateWithFlags(&c->side_spec, cudaStreamNonBlocking));
  A(cudaStreamCreateWithFlags(&c->side_ema, cudaStreamNonBlocking));
  A(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
  A(cudaEventCreateWithFlags(&c->ev_spec, cudaEventDisableTiming));
  A(cudaEventCreateWithFlags(&c->ev_sel, cudaEventDisableTiming));
  c->ev_upd.assign(c->NL, nullptr);
  c->upd_pending.assign(c->NL, 0);
  c->bud_eff.assign(c->NL, c->Bud);
  c->bud_seq_h.assign((size_t)c->NL * c->maxB, 0);
  c->kscale.assign(c->NL, nullptr); c->vscale.assign(c->NL, nullptr);
  for (int l = 0; l < c->NL; ++l) A(cudaEventCreateWithFlags(&c->ev_upd[l], cudaEventDisableTiming));
  if (e != cudaSuccess) {
    g_create_err = std::string("prr_create: ") + cudaGetErrorString(e);
    const bool nomem = e == cudaErrorMemoryAllocation;
    cudaGetLastError();
    prr_destroy(c);
    return nomem ? PRR_E_NOMEM : PRR_E_CUDA;
  }
  *out = c;
  return PRR_OK;
}

extern "C" int32_t prr_destroy(prr_ctx* c) {
  if (!c) return PRR_E_INVALID;
  cudaDeviceSynchronize();
  for (void* p : c->allocs) cudaFree(p);
  if (c->st_pin) cudaFreeHost(c->st_pin);
  if (c->st_out_h) cudaFreeHost(c->st_out_h);
  if (c->done_h) cudaFreeHost((void*)c->done_h);
  if (c->tl) cudaFreeHost(c->tl);
  if (c->cal_state) cudaFree(c->cal_state);
  if (c->cal_mask) cudaFree(c->cal_mask);
  if (c->cal_den) cudaFree(c->cal_den);
  if (c->side_spec) cudaStreamDestroy(c->side_spec);
  if (c->side_ema) cudaStreamDestroy(c->side_ema);
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_spec) cudaEventDestroy(c->ev_spec);
  if (c->ev_sel) cudaEventDestroy(c->ev_sel);
  for (cudaEvent_t ev : c->ev_upd) if (ev) cudaEventDestroy(ev);
  cudaGetLastError();
  delete c;
  return PRR_OK;
}

// ---------------------------------------------------------------------------------------------
static int check_kv(prr_ctx* c, const prr_paged_kv* kv, const char* fn) {
  if (!c) return PRR_E_INVALID;
  if (!kv) PRR_FAIL(c, PRR_E_INVALID, "%s: null prr_paged_kv", fn);
  if (!kv->k_pages || !kv->v_pages || !kv->block_table || !kv->seq_lens)
    PRR_FAIL(c, PRR_E_INVALID, "%s: null pointer in prr_paged_kv", fn);
  if (!aligned16(kv->k_pages) || !aligned16(kv->v_pages))
    PRR_FAIL(c, PRR_E_INVALID, "%s: k_pages / v_pages must be 16-byte aligned", fn);
  if (kv->batch < 1 || kv->batch > c->maxB) PRR_FAIL(c, PRR_E_INVALID, "%s: batch out of range", fn);
  if (kv->layer < 0 || kv->layer >= c->NL) PRR_FAIL(c, PRR_E_INVALID, "%s: layer out of range", fn);
  if (c->lay.kv_dtype == PRR_FP8_E4M3 && (!c->kscale[kv->layer] || !c->vscale[kv->layer]))
    PRR_FAIL(c, PRR_E_STATE, "%s: fp8 KV: call prr_set_kv_scales for layer %d first", fn, kv->layer);
  return PRR_OK;
}
#define NO_FP8(fn) do { if (ctx && ctx->lay.kv_dtype == PRR_FP8_E4M3) \
    PRR_FAIL(ctx, PRR_E_UNSUPPORTED, "%s: not available with PRR_FP8_E4M3 (a token cannot join a block quantised with a fixed scale)", fn); } while (0)
#define CHECK_KV(fn) do { int _r = check_kv(ctx, kv, fn); if (_r) return _r; } while (0)
#define CHECK_PTR(p, fn) do { if (!(p)) PRR_FAIL(ctx, PRR_E_INVALID, "%s: null %s", fn, #p); \
    if (!aligned16(p)) PRR_FAIL(ctx, PRR_E_INVALID, "%s: %s must be 16-byte aligned", fn, #p); } while (0)

// Make `s` wait for every EMA update still running on the side stream.
static void join_updates(prr_ctx* c, cudaStream_t s) {
  for (int l = 0; l < c->NL; ++l)
    if (c->upd_pending[l]) { cudaStreamWaitEvent(s, c->ev_upd[l], 0); c->upd_pending[l] = 0; }
}
static void join_layer(prr_ctx* c, int layer, cudaStream_t s) {
  if (c->upd_pending[layer]) { cudaStreamWaitEvent(s, c->ev_upd[layer], 0); c->upd_pending[layer] = 0; }
}

extern "C" int32_t prr_build_summaries(prr_ctx* ctx, const prr_paged_kv* kv, void* summaries, void* stream) {
  CHECK_KV("prr_build_summaries");
  CHECK_PTR(summaries, "prr_build_summaries");
  launch_build_summaries(ctx, kv, summaries, (cudaStream_t)stream);
  return check_launch(ctx, "prr_build_summaries");
}

extern "C" int32_t prr_append(prr_ctx* ctx, const prr_paged_kv* kv, const void* k_new, const void* v_new,
                              void* summaries, void* stream) {
  NO_FP8("prr_append");
  CHECK_KV("prr_append");
  CHECK_PTR(k_new, "prr_append"); CHECK_PTR(v_new, "prr_append"); CHECK_PTR(summaries, "prr_append");
  // (PRR_STREAMS: the layer's EMA update on the side stream derives the block count from seq_lens, which
  // this call increments: it must have finished)
  join_layer(ctx, kv->layer, (cudaStream_t)stream);
  launch_append(ctx, kv, k_new, v_new, summaries, (cudaStream_t)stream);
  return check_launch(ctx, "prr_append");
}

extern "C" int32_t prr_quantize_kv_fp8(prr_ctx* ctx, const prr_paged_kv* kv, void* k8_pages, void* v8_pages,
                                       float* k_scale, float* v_scale, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (!kv || !kv->k_pages || !kv->v_pages || !kv->block_table || !kv->seq_lens)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_quantize_kv_fp8: null pointer in prr_paged_kv");
  if (kv->batch < 1 || kv->batch > ctx->maxB) PRR_FAIL(ctx, PRR_E_INVALID, "prr_quantize_kv_fp8: batch out of range");
  if (!k8_pages || !v8_pages || !k_scale || !v_scale) PRR_FAIL(ctx, PRR_E_INVALID, "prr_quantize_kv_fp8: null output");
  if (!aligned16(k8_pages) || !aligned16(v8_pages)) PRR_FAIL(ctx, PRR_E_INVALID, "prr_quantize_kv_fp8: pages must be 16-byte aligned");
  launch_quantize_fp8(ctx, kv, k8_pages, v8_pages, k_scale, v_scale, (cudaStream_t)stream);
  return check_launch(ctx, "prr_quantize_kv_fp8");
}

extern "C" int32_t prr_set_kv_scales(prr_ctx* ctx, int32_t layer, const float* k_scale, const float* v_scale) {
  if (!ctx) return PRR_E_INVALID;
  if (ctx->lay.kv_dtype != PRR_FP8_E4M3) PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_kv_scales: the ctx was not created with PRR_FP8_E4M3");
  if (layer < 0 || layer >= ctx->NL) PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_kv_scales: layer out of range");
  if (!k_scale || !v_scale) PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_kv_scales: null argument");
  ctx->kscale[layer] = k_scale; ctx->vscale[layer] = v_scale;
  return PRR_OK;
}

// ---------------------------------------------------------------------------------------------
__global__ void k_set_theta(double* theta, int n, double a, double b, double g) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { theta[i * 3] = a; theta[i * 3 + 1] = b; theta[i * 3 + 2] = g; }
}
__global__ void k_fill_i32(int32_t* p, size_t n, int32_t v) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// Fused orchestration keeps the prediction in two buffers selected by a device-side parity.
// which = 0: the buffer the NEXT step reads; which = 1: the buffer the LAST step read.
__global__ void k_copy_P(int32_t* P0, int32_t* P1, const int32_t* parity, int which, int32_t* other,
                         size_t n, int to_pbuf) {
  int32_t* P = ((*parity ^ which) & 1) ? P1 : P0;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { if (to_pbuf) P[i] = other[i]; else other[i] = P[i]; }
}
// After a stage-level prediction landed in P_next: make it the one the next fused step reads.
static void sync_pred(prr_ctx* c, int layer, int seq0, int nseq, cudaStream_t s) {
  if (!c->fused || c->Bud <= 0) return;
  const size_t off = (layer_rows(c, layer) + (size_t)seq0 * c->Hkv) * c->Bud;
  const size_t n = (size_t)nseq * c->Hkv * c->Bud;
  k_copy_P<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(c->Pbuf[0] + off, c->Pbuf[1] + off,
                                                       c->parity + layer, 0, c->P_next + off, n, 1);
  c->launches++;
}

extern "C" int32_t prr_set_ema_params(prr_ctx* ctx, int32_t layer, int32_t seq, double alpha, double beta,
                                      double gamma, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || seq < -1 || seq >= ctx->maxB)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_ema_params: layer/seq out of range");
  if (!(alpha > 0.0 && alpha <= 1.0 && beta > 0.0 && beta <= 1.0 && gamma >= 0.0 && gamma <= 1.0))
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_ema_params: need alpha,beta in (0,1], gamma in [0,1] (PAPER.md:149,156)");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  const int n = seq < 0 ? ctx->maxB : 1;
  double* th = ctx->theta + ((size_t)layer * ctx->maxB + (seq < 0 ? 0 : seq)) * 3;
  k_set_theta<<<(n + 63) / 64, 64, 0, s>>>(th, n, alpha, beta, gamma);
  ctx->launches++;
  return check_launch(ctx, "prr_set_ema_params");
}

extern "C" int32_t prr_reset_ema(prr_ctx* ctx, int32_t layer, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL) PRR_FAIL(ctx, PRR_E_INVALID, "prr_reset_ema: layer out of range");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  const size_t r = layer_rows(ctx, layer), n = (size_t)ctx->maxB * ctx->Hkv;
  PRR_CUDA(ctx, cudaMemsetAsync(ctx->n_state + r, 0, n * sizeof(int32_t), s));
  if (ctx->Bud > 0)
    PRR_CUDA(ctx, cudaMemsetAsync(ctx->P_next + r * ctx->Bud, 0xff, n * ctx->Bud * sizeof(int32_t), s));
  if (ctx->Bud > 0 && ctx->fused) {
    PRR_CUDA(ctx, cudaMemsetAsync(ctx->Pbuf[0] + r * ctx->Bud, 0xff, n * ctx->Bud * sizeof(int32_t), s));
    PRR_CUDA(ctx, cudaMemsetAsync(ctx->Pbuf[1] + r * ctx->Bud, 0xff, n * ctx->Bud * sizeof(int32_t), s));
  }
  return PRR_OK;
}

extern "C" int32_t prr_calibrate(prr_ctx* ctx, int32_t layer, int32_t seq, const float* prefill_scores,
                                 int32_t T, int32_t N, const int32_t* n_valid, double* theta_out,
                                 double* H_out, double* H_all_out, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || seq < 0 || seq >= ctx->maxB)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_calibrate: layer/seq out of range");
  if (!prefill_scores) PRR_FAIL(ctx, PRR_E_INVALID, "prr_calibrate: null prefill_scores");
  if (T < 1 || N < 1 || N > ctx->MB) PRR_FAIL(ctx, PRR_E_INVALID, "prr_calibrate: need T >= 1 and 1 <= N <= max_blocks_per_seq");
  cudaStream_t s = (cudaStream_t)stream;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(s, &cap);
  if (cap != cudaStreamCaptureStatusNone) PRR_FAIL(ctx, PRR_E_STATE, "prr_calibrate: cannot run inside a stream capture");
  join_layer(ctx, layer, s);
  int r = launch_calibrate(ctx, layer, seq, prefill_scores, T, N, n_valid, s);
  if (r) return r;
  if ((r = check_launch(ctx, "prr_calibrate"))) return r;
  if (ctx->Bud > 0) {  // first decode step's prediction (Q5)
    EmaArgs e{};
    e.layer = layer; e.batch = 1; e.seq0 = seq;
    const size_t rows = layer_rows(ctx, layer) + (size_t)seq * ctx->Hkv;
    e.P_out = ctx->P_next + rows * ctx->Bud;
    launch_ema(ctx, e, s);
    sync_pred(ctx, layer, seq, 1, s);
    if ((r = check_launch(ctx, "prr_calibrate(predict)"))) return r;
  }
  if (theta_out || H_out || H_all_out) {
    double H[80];
    int32_t best = 0;
    double* dH = ctx->cal_acc + 2 * 80 * ctx->Hkv;
    PRR_CUDA(ctx, cudaMemcpyAsync(H, dH, sizeof(H), cudaMemcpyDeviceToHost, s));
    PRR_CUDA(ctx, cudaMemcpyAsync(&best, dH + 80, sizeof(best), cudaMemcpyDeviceToHost, s));
    double th[3];
    PRR_CUDA(ctx, cudaMemcpyAsync(th, ctx->theta + ((size_t)layer * ctx->maxB + seq) * 3, sizeof(th),
                                  cudaMemcpyDeviceToHost, s));
    PRR_CUDA(ctx, cudaStreamSynchronize(s));
    if (theta_out) memcpy(theta_out, th, sizeof(th));
    if (H_out) *H_out = H[best];
    if (H_all_out) memcpy(H_all_out, H, sizeof(H));
  }
  return PRR_OK;
}

extern "C" int32_t prr_predict(prr_ctx* ctx, int32_t layer, int32_t batch, int32_t* P_out,
                               int32_t* count_out, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || batch < 1 || batch > ctx->maxB)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_predict: layer/batch out of range");
  if (!P_out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_predict: null P_out");
  if (ctx->Bud < 1) PRR_FAIL(ctx, PRR_E_STATE, "prr_predict: ctx was created with budget 0");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  EmaArgs e{};
  e.layer = layer; e.batch = batch; e.seq0 = 0;
  e.P_out = P_out; e.P_count = count_out;
  launch_ema(ctx, e, s);
  return check_launch(ctx, "prr_predict");
}

extern "C" int32_t prr_ema_update(prr_ctx* ctx, int32_t layer, int32_t batch, const float* scores,
                                  const int32_t* n_blocks, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || batch < 1 || batch > ctx->maxB)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_ema_update: layer/batch out of range");
  if (!scores || !n_blocks) PRR_FAIL(ctx, PRR_E_INVALID, "prr_ema_update: null argument");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  EmaArgs e{};
  e.layer = layer; e.batch = batch; e.seq0 = 0;
  e.scores = scores; e.n_blocks = n_blocks;
  e.P_out = ctx->P_next + layer_rows(ctx, layer) * ctx->Bud;
  launch_ema(ctx, e, s);
  sync_pred(ctx, layer, 0, batch, s);
  return check_launch(ctx, "prr_ema_update");
}

// ---------------------------------------------------------------------------------------------
// Profiling-guided speculation budget (PAPER.md:204-208 section 4.4, :229, :424 A.6)
// ---------------------------------------------------------------------------------------------
static void repredict(prr_ctx* c, int layer, cudaStream_t s) {  // P of the next step under the layer's current budget
  if (c->Bud <= 0) return;
  join_layer(c, layer, s);
  EmaArgs e{};
  e.layer = layer; e.batch = c->maxB; e.seq0 = 0;
  e.P_out = c->P_next + layer_rows(c, layer) * c->Bud;
  launch_ema(c, e, s);
  sync_pred(c, layer, 0, c->maxB, s);
}

__global__ void k_set_i32(int32_t* p, int32_t v) { *p = v; }

extern "C" int32_t prr_set_budget_seq(prr_ctx* ctx, int32_t layer, int32_t seq, int32_t budget, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || seq < 0 || seq >= ctx->maxB) PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_budget_seq: layer / seq out of range");
  if (budget < -1 || budget > ctx->Bud) PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_budget_seq: budget must be -1 (the layer's) or 0 .. the budget of prr_create");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  const size_t i = (size_t)layer * ctx->maxB + seq;
  ctx->bud_seq_h[i] = budget + 1;
  k_set_i32<<<1, 1, 0, s>>>(ctx->bud_seq + i, budget + 1);
  ctx->launches++;
  repredict(ctx, layer, s);  // the next decode step already speculates on the new budget
  return check_launch(ctx, "prr_set_budget_seq");
}

extern "C" int32_t prr_get_budget_seq(const prr_ctx* ctx, int32_t layer, int32_t seq, int32_t* budget_out) {
  if (!ctx || !budget_out) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || seq < 0 || seq >= ctx->maxB) return PRR_E_INVALID;
  const int v = ctx->bud_seq_h[(size_t)layer * ctx->maxB + seq];
  *budget_out = v > 0 ? v - 1 : ctx->bud_eff[layer];
  return PRR_OK;
}

extern "C" int32_t prr_set_mode(prr_ctx* ctx, int32_t mode, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (mode != PRR_MODE_S3 && mode != PRR_MODE_S2 && mode != PRR_MODE_S1) PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_mode: unknown mode");
  if (mode == PRR_MODE_S1 && (ctx->lay.overpredict_policy != PRR_DROP || !ctx->fused))
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_mode: S1 (recompute on any miss) needs PRR_DROP and PRR_FUSED");
  ctx->mode = mode;
  if (mode == PRR_MODE_S3) return PRR_OK;
  cudaStream_t s = (cudaStream_t)stream;
  for (int l = 0; l < ctx->NL; ++l) {  // "reuse the last step's top-K": alpha = beta = 1, gamma = 0, |P| = K
    join_layer(ctx, l, s);
    k_set_theta<<<(ctx->maxB + 63) / 64, 64, 0, s>>>(ctx->theta + (size_t)l * ctx->maxB * 3, ctx->maxB, 1.0, 1.0, 0.0);
    ctx->launches++;
    ctx->bud_eff[l] = std::min(ctx->K, ctx->Bud);
    repredict(ctx, l, s);
  }
  return check_launch(ctx, "prr_set_mode");
}

extern "C" int32_t prr_set_budget(prr_ctx* ctx, int32_t layer, int32_t budget, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < -1 || layer >= ctx->NL || budget < 0 || budget > ctx->Bud)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_budget: need -1 <= layer < n_layers and 0 <= budget <= the budget of prr_create");
  for (int l = layer < 0 ? 0 : layer; l < (layer < 0 ? ctx->NL : layer + 1); ++l) {
    ctx->bud_eff[l] = budget;
    repredict(ctx, l, (cudaStream_t)stream);
  }
  return check_launch(ctx, "prr_set_budget");
}

extern "C" int32_t prr_get_budget(const prr_ctx* ctx, int32_t layer, int32_t* budget_out) {
  if (!ctx || !budget_out || layer < 0 || layer >= ctx->NL) return PRR_E_INVALID;
  *budget_out = ctx->bud_eff[layer];
  return PRR_OK;
}

extern "C" int32_t prr_profile_budget(prr_ctx* ctx, const prr_paged_kv* kv, const void* q_traj, int32_t T,
                                      const void* summaries, const int32_t* budgets, int32_t n_budgets,
                                      int32_t cold_l2, float* us_out, float* us_sequential_out,
                                      int32_t* best_budget_out, void* stream) {
  CHECK_KV("prr_profile_budget");
  CHECK_PTR(q_traj, "prr_profile_budget"); CHECK_PTR(summaries, "prr_profile_budget");
  if (T < 2 || n_budgets < 1 || !budgets) PRR_FAIL(ctx, PRR_E_INVALID, "prr_profile_budget: need T >= 2 and at least one budget");
  for (int i = 0; i < n_budgets; ++i)
    if (budgets[i] < 0 || budgets[i] > ctx->Bud) PRR_FAIL(ctx, PRR_E_INVALID, "prr_profile_budget: budget out of range");
  cudaStream_t s = (cudaStream_t)stream;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(s, &cap);
  if (cap != cudaStreamCaptureStatusNone) PRR_FAIL(ctx, PRR_E_STATE, "prr_profile_budget: cannot run inside a stream capture");
  join_updates(ctx, s);
  PRR_CUDA(ctx, cudaStreamSynchronize(s));
  const int layer = kv->layer;
  const size_t r = layer_rows(ctx, layer), nr = (size_t)ctx->maxB * ctx->Hkv;
  // the layer's predictor state is saved and put back: profiling leaves no trace
  struct Save { void* dev; void* copy; size_t bytes; };
  std::vector<Save> saves = {
      {ctx->ema_l + r * ctx->MB, nullptr, nr * ctx->MB * sizeof(double)}, {ctx->ema_v + r * ctx->MB, nullptr, nr * ctx->MB * sizeof(double)},
      {ctx->n_state + r, nullptr, nr * sizeof(int32_t)}, {ctx->parity + layer, nullptr, sizeof(int32_t)},
      {ctx->Pbuf[0] + r * ctx->Bud, nullptr, nr * ctx->Bud * sizeof(int32_t)}, {ctx->Pbuf[1] + r * ctx->Bud, nullptr, nr * ctx->Bud * sizeof(int32_t)},
      {ctx->P_next + r * ctx->Bud, nullptr, nr * ctx->Bud * sizeof(int32_t)}, {ctx->P_used + r * ctx->Bud, nullptr, nr * ctx->Bud * sizeof(int32_t)},
      {ctx->stats, nullptr, 4 * sizeof(unsigned long long)}};
  cudaError_t e = cudaSuccess;
  for (auto& v : saves) {
    if (!v.bytes) continue;
    if (e == cudaSuccess) e = cudaMalloc(&v.copy, v.bytes);
    if (e == cudaSuccess) e = cudaMemcpyAsync(v.copy, v.dev, v.bytes, cudaMemcpyDeviceToDevice, s);
  }
  void* flush = nullptr;
  const size_t flush_bytes = (size_t)256 << 20;  // larger than L2
  if (cold_l2 && e == cudaSuccess) e = cudaMalloc(&flush, flush_bytes);
  std::vector<cudaEvent_t> ev(2 * (size_t)T, nullptr);
  for (auto& x : ev) if (e == cudaSuccess) e = cudaEventCreate(&x);
  const int saved_budget = ctx->bud_eff[layer];
  const size_t qstep = (size_t)kv->batch * ctx->Hq * ctx->D;  // bf16 elements per step
  int rc = PRR_OK;
  auto restore = [&]() { for (auto& v : saves) if (v.copy) cudaMemcpyAsync(v.dev, v.copy, v.bytes, cudaMemcpyDeviceToDevice, s); };
  auto run = [&](int budget, bool sequential, float* us) {  // mean over the steps after the first (warm-up of clocks and code)
    restore();
    ctx->bud_eff[layer] = budget;
    repredict(ctx, layer, s);
    for (int t = 0; t < T && rc == PRR_OK; ++t) {
      if (flush) cudaMemsetAsync(flush, t, flush_bytes, s);
      cudaEventRecord(ev[2 * t], s);
      const void* q = (const uint16_t*)q_traj + (size_t)t * qstep;
      rc = sequential ? prr_attend(ctx, kv, q, summaries, ctx->st_out, stream) : prr_decode_step(ctx, kv, q, summaries, ctx->st_out, stream);
      join_layer(ctx, layer, s);
      cudaEventRecord(ev[2 * t + 1], s);
    }
    if (rc != PRR_OK) return;
    if (cudaStreamSynchronize(s) != cudaSuccess) { rc = PRR_E_CUDA; return; }
    std::vector<float> v;  // the MEDIAN step: one slow step (a page fault, another tenant) must not decide a budget
    for (int t = 1; t < T; ++t) { float ms = 0.f; cudaEventElapsedTime(&ms, ev[2 * t], ev[2 * t + 1]); v.push_back(ms); }
    std::sort(v.begin(), v.end());
    *us = v[v.size() / 2] * 1e3f;
  };
  float best_us = 0.f, seq_us = 0.f;
  (void)best_us;
  int best = 0;
  if (e == cudaSuccess) {
    run(0, true, &seq_us);
    // No speculation at all is the fallback PRR must beat, and "safe" is read with a
    // margin: a budget is taken only if it beats the sequential path by more than 2 % (differences below that are
    // run-to-run noise of the sweep, and a wrong "yes" costs bandwidth on every step).
    // Among the budgets that are safe, the LARGEST one within 1 % of the fastest is taken ("largest safe
    // delta": a larger prediction costs nothing while it hides behind selection, and it raises the hit rate).
    std::vector<float> uss(n_budgets, 0.f);
    float min_us = seq_us * 0.98f;
    best = 0;
    for (int i = 0; i < n_budgets && rc == PRR_OK; ++i) {
      run(budgets[i], false, &uss[i]);
      if (us_out) us_out[i] = uss[i];
      if (rc == PRR_OK && budgets[i] > 0 && uss[i] < min_us) min_us = uss[i];
    }
    for (int i = 0; i < n_budgets && rc == PRR_OK; ++i)
      if (budgets[i] > best && uss[i] < seq_us * 0.98f && uss[i] <= min_us * 1.01f) best = budgets[i];
    best_us = min_us;
    restore();
    ctx->bud_eff[layer] = saved_budget;
    repredict(ctx, layer, s);
    cudaStreamSynchronize(s);
  }
  for (auto& x : ev) if (x) cudaEventDestroy(x);
  for (auto& v : saves) if (v.copy) cudaFree(v.copy);
  if (flush) cudaFree(flush);
  if (e != cudaSuccess) { cudaGetLastError(); PRR_FAIL(ctx, e == cudaErrorMemoryAllocation ? PRR_E_NOMEM : PRR_E_CUDA, "prr_profile_budget: %s", cudaGetErrorString(e)); }
  if (rc != PRR_OK) return rc;
  if (us_sequential_out) *us_sequential_out = seq_us;
  if (best_budget_out) *best_budget_out = best;
  return check_launch(ctx, "prr_profile_budget");
}

// Least-squares polynomial budget(context length) through the profiled points ("polynomial
// regression" for lengths off the grid).  Normal equations in x = len / max(len), Gaussian elimination.
extern "C" int32_t prr_budget_fit(prr_ctx* ctx, int32_t n, const int32_t* ctx_lens, const int32_t* budgets, int32_t degree) {
  if (!ctx) return PRR_E_INVALID;
  if (n < 1 || !ctx_lens || !budgets || degree < 0 || degree > 3) PRR_FAIL(ctx, PRR_E_INVALID, "prr_budget_fit: need n >= 1 points and 0 <= degree <= 3");
  const int m = std::min(degree, n - 1) + 1;  // coefficients
  double xs = 1.0;
  for (int i = 0; i < n; ++i) { if (ctx_lens[i] < 1) PRR_FAIL(ctx, PRR_E_INVALID, "prr_budget_fit: context lengths must be >= 1"); xs = std::max(xs, (double)ctx_lens[i]); }
  double A[4][5] = {};
  for (int i = 0; i < n; ++i) {
    const double x = ctx_lens[i] / xs;
    double p[7] = {1, x, x * x, x * x * x, x * x * x * x, x * x * x * x * x, x * x * x * x * x * x};
    for (int a = 0; a < m; ++a) { for (int b = 0; b < m; ++b) A[a][b] += p[a + b]; A[a][m] += p[a] * budgets[i]; }
  }
  for (int c0 = 0; c0 < m; ++c0) {
    int piv = c0;
    for (int rr = c0 + 1; rr < m; ++rr) if (std::fabs(A[rr][c0]) > std::fabs(A[piv][c0])) piv = rr;
    if (std::fabs(A[piv][c0]) < 1e-12) PRR_FAIL(ctx, PRR_E_INVALID, "prr_budget_fit: the points do not determine a polynomial of this degree");
    for (int b = 0; b <= m; ++b) std::swap(A[c0][b], A[piv][b]);
    for (int rr = 0; rr < m; ++rr) {
      if (rr == c0) continue;
      const double f = A[rr][c0] / A[c0][c0];
      for (int b = c0; b <= m; ++b) A[rr][b] -= f * A[c0][b];
    }
  }
  ctx->bud_poly.assign(m, 0.0);
  for (int a = 0; a < m; ++a) ctx->bud_poly[a] = A[a][m] / A[a][a];
  ctx->bud_xscale = xs;
  return PRR_OK;
}

extern "C" int32_t prr_budget_for(const prr_ctx* ctx, int32_t ctx_len, int32_t* budget_out) {
  if (!ctx || !budget_out || ctx_len < 0) return PRR_E_INVALID;
  if (ctx->bud_poly.empty()) { *budget_out = ctx->Bud; return PRR_OK; }  // nothing fitted: the budget of prr_create
  const double x = ctx_len / ctx->bud_xscale;
  double y = 0.0;
  for (size_t a = ctx->bud_poly.size(); a-- > 0;) y = y * x + ctx->bud_poly[a];
  const long v = std::lround(y);
  *budget_out = (int32_t)std::min<long>(ctx->Bud, std::max<long>(0, v));
  return PRR_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" int32_t prr_score(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* summaries,
                             float* scores_out, void* stream) {
  CHECK_KV("prr_score");
  CHECK_PTR(q, "prr_score"); CHECK_PTR(summaries, "prr_score");
  if (!scores_out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_score: null scores_out");
  launch_score(ctx, kv, q, summaries, scores_out, (cudaStream_t)stream);
  return check_launch(ctx, "prr_score");
}

extern "C" int32_t prr_topk(prr_ctx* ctx, const float* scores, const int32_t* n_blocks, int32_t batch,
                            int32_t k, int32_t* idx_out, int32_t* count_out, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (!scores || !n_blocks || !idx_out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_topk: null argument");
  if (batch < 1 || batch > ctx->maxB || k < 1 || k > 1024)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_topk: need 1 <= batch <= max_batch, 1 <= k <= 1024");
  SelectArgs a{};
  a.scores = scores; a.row_stride = ctx->MB; a.n_blocks = n_blocks; a.bs = ctx->bs;
  a.batch = batch; a.Hkv = ctx->Hkv; a.k = k; a.A_out = idx_out; a.A_count = count_out;
  launch_select(ctx, a, (cudaStream_t)stream);
  return check_launch(ctx, "prr_topk");
}

extern "C" int32_t prr_speculate(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const int32_t* P,
                                 float* O_part, float* m_part, float* l_part, void* stream) {
  CHECK_KV("prr_speculate");
  if (ctx->bs > 128) PRR_FAIL(ctx, PRR_E_UNSUPPORTED, "prr_speculate: blocks of 256 tokens run on the fused step only");
  CHECK_PTR(q, "prr_speculate");
  if (!P || !O_part || !m_part || !l_part) PRR_FAIL(ctx, PRR_E_INVALID, "prr_speculate: null argument");
  if (ctx->Bud < 1) PRR_FAIL(ctx, PRR_E_STATE, "prr_speculate: ctx was created with budget 0");
  launch_partial(ctx, kv, q, P, ctx->Bud, O_part, m_part, l_part, (cudaStream_t)stream);
  return check_launch(ctx, "prr_speculate");
}

extern "C" int32_t prr_repair(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const int32_t* A,
                              const int32_t* P, const float* O_part, const float* m_part,
                              const float* l_part, float* out, float* m_out, float* l_out, void* stream) {
  CHECK_KV("prr_repair");
  if (ctx->bs > 128) PRR_FAIL(ctx, PRR_E_UNSUPPORTED, "prr_repair: blocks of 256 tokens run on the fused step only");
  CHECK_PTR(q, "prr_repair");
  if (!A || !out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_repair: null argument");
  if (P && (!O_part || !m_part || !l_part)) PRR_FAIL(ctx, PRR_E_INVALID, "prr_repair: P given without its partial states");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t r = layer_rows(ctx, kv->layer);
  SelectArgs a{};
  a.scores = nullptr; a.row_stride = ctx->MB; a.seq_lens = kv->seq_lens; a.bs = ctx->bs;
  a.batch = kv->batch; a.Hkv = ctx->Hkv; a.k = ctx->K;
  a.A_out = const_cast<int32_t*>(A);  // read-only in this mode
  a.P = P; a.Bud = ctx->Bud;
  a.M_out = ctx->setM + r * ctx->K;
  a.merge_src = ctx->merge_src; a.merge_n = ctx->merge_n;
  a.counts = ctx->counts + r * 3;
  a.retain = ctx->lay.overpredict_policy == PRR_RETAIN;
  launch_select(ctx, a, s);
  launch_partial(ctx, kv, q, a.M_out, ctx->K, ctx->O_rep, ctx->m_rep, ctx->l_rep, s);
  launch_merge(ctx, kv->batch, ctx->merge_src, ctx->merge_n, O_part, m_part, l_part, ctx->Bud,
               ctx->O_rep, ctx->m_rep, ctx->l_rep, ctx->K, out, m_out, l_out, s);
  return check_launch(ctx, "prr_repair");
}

// ---------------------------------------------------------------------------------------------
static void enqueue_ema(prr_ctx* c, const prr_paged_kv* kv, cudaStream_t main, bool wait_spec) {
  // Off the critical path: Eq. 3 update with this step's scores, then the next step's P.  It must
  // not overwrite P while the speculative launch and the diff still read it.
  const size_t r = layer_rows(c, kv->layer);
  cudaEventRecord(c->ev_sel, main);
  cudaStreamWaitEvent(c->side_ema, c->ev_sel, 0);
  if (wait_spec) cudaStreamWaitEvent(c->side_ema, c->ev_spec, 0);
  EmaArgs e{};
  e.layer = kv->layer; e.batch = kv->batch; e.seq0 = 0;
  e.scores = c->scores + r * c->MB;
  e.seq_lens = kv->seq_lens;
  e.P_out = c->P_next + r * c->Bud;
  e.P_save = c->Bud > 0 ? c->P_used + r * c->Bud : nullptr;
  launch_ema(c, e, c->side_ema);
  cudaEventRecord(c->ev_upd[kv->layer], c->side_ema);
  c->upd_pending[kv->layer] = 1;
}

static int fused_step(prr_ctx* c, const prr_paged_kv* kv, const void* q, const void* summaries,
                      float* out, int spec, cudaStream_t s, const char* fn, const void* k_new = nullptr,
                      const void* v_new = nullptr) {
  // Which fused kernel: the persistent cooperative grid when the rows are few (its warps are spread over
  // every SM whatever the batch), a cluster per row once the rows fill the GPU (measured: DESIGN.md section 8).
  const int rows = kv->batch * c->Hkv;
  // a run-time budget of 0 (prr_set_budget re-predicted: P is empty) IS the sequential path: take it outright
  if (spec && c->bud_eff[kv->layer] == 0) {
    bool any = false;  // (a sequence with its own budget > 0 still speculates)
    for (int b = 0; b < kv->batch; ++b) any |= c->bud_seq_h[(size_t)kv->layer * c->maxB + b] > 1;
    if (!any) spec = 0;
  }
  int kern = c->kernel;
  if (kern == 0) kern = rows >= 64 ? 2 : 1;
  if (c->bs > 128 || c->mode == PRR_MODE_S1) kern = 2;  // (only the cluster kernel cuts a block into sub-tiles / recomputes on a miss)
  if (kern == 1 && !c->coop) kern = 2;
  c->last_kernel = kern;
  const int e = kern == 2 ? launch_step_cluster(c, kv, q, summaries, out, spec, s, k_new, v_new)
                          : launch_step_persist(c, kv, q, summaries, out, spec, s, k_new, v_new);
  if (e) {
    cudaGetLastError();
    PRR_FAIL(c, PRR_E_CUDA, "%s: fused step launch: %s", fn, cudaGetErrorString((cudaError_t)e));
  }
  return check_launch(c, fn);
}

extern "C" int32_t prr_attend(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* summaries,
                              float* out, void* stream) {
  CHECK_KV("prr_attend");
  CHECK_PTR(q, "prr_attend"); CHECK_PTR(summaries, "prr_attend");
  if (!out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_attend: null out");
  cudaStream_t s = (cudaStream_t)stream;
  if (ctx->fused) return fused_step(ctx, kv, q, summaries, out, 0, s, "prr_attend");
  const size_t r = layer_rows(ctx, kv->layer);
  join_layer(ctx, kv->layer, s);
  float* sc = ctx->scores + r * ctx->MB;
  launch_score(ctx, kv, q, summaries, sc, s);
  SelectArgs a{};
  a.scores = sc; a.row_stride = ctx->MB; a.seq_lens = kv->seq_lens; a.bs = ctx->bs;
  a.batch = kv->batch; a.Hkv = ctx->Hkv; a.k = ctx->K;
  a.A_out = ctx->setA + r * ctx->K;
  a.P = nullptr; a.Bud = ctx->Bud;
  a.M_out = ctx->setM + r * ctx->K;
  a.merge_src = ctx->merge_src; a.merge_n = ctx->merge_n;
  a.counts = ctx->counts + r * 3;
  a.retain = 0;
  launch_select(ctx, a, s);
  enqueue_ema(ctx, kv, s, false);
  launch_partial(ctx, kv, q, a.M_out, ctx->K, ctx->O_rep, ctx->m_rep, ctx->l_rep, s);
  launch_merge(ctx, kv->batch, ctx->merge_src, ctx->merge_n, ctx->O_spec, ctx->m_spec, ctx->l_spec,
               ctx->Bud, ctx->O_rep, ctx->m_rep, ctx->l_rep, ctx->K, out, nullptr, nullptr, s);
  return check_launch(ctx, "prr_attend");
}

extern "C" int32_t prr_decode_step(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* summaries,
                                   float* out, void* stream) {
  CHECK_KV("prr_decode_step");
  CHECK_PTR(q, "prr_decode_step"); CHECK_PTR(summaries, "prr_decode_step");
  if (!out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_decode_step: null out");
  cudaStream_t s = (cudaStream_t)stream;
  if (ctx->fused) return fused_step(ctx, kv, q, summaries, out, 1, s, "prr_decode_step");
  const size_t r = layer_rows(ctx, kv->layer);
  const bool spec = ctx->Bud > 0;
  join_layer(ctx, kv->layer, s);  // this layer's previous EMA update / prediction must be complete
  const int32_t* P = spec ? ctx->P_next + r * ctx->Bud : nullptr;
  if (spec) {
    // speculation branch: attention over the predicted blocks while selection is in flight
    cudaEventRecord(ctx->ev_fork, s);
    cudaStreamWaitEvent(ctx->side_spec, ctx->ev_fork, 0);
    launch_partial(ctx, kv, q, P, ctx->Bud, ctx->O_spec, ctx->m_spec, ctx->l_spec, ctx->side_spec);
    cudaEventRecord(ctx->ev_spec, ctx->side_spec);
  }
  // selection branch (critical path): score -> top-K + diff -> repair partials of A\P
  float* sc = ctx->scores + r * ctx->MB;
  launch_score(ctx, kv, q, summaries, sc, s);
  SelectArgs a{};
  a.scores = sc; a.row_stride = ctx->MB; a.seq_lens = kv->seq_lens; a.bs = ctx->bs;
  a.batch = kv->batch; a.Hkv = ctx->Hkv; a.k = ctx->K;
  a.A_out = ctx->setA + r * ctx->K;
  a.P = P; a.Bud = ctx->Bud;
  a.M_out = ctx->setM + r * ctx->K;
  a.merge_src = ctx->merge_src; a.merge_n = ctx->merge_n;
  a.counts = ctx->counts + r * 3;
  a.stats = ctx->stats;
  a.retain = ctx->lay.overpredict_policy == PRR_RETAIN;
  launch_select(ctx, a, s);
  enqueue_ema(ctx, kv, s, spec);
  launch_partial(ctx, kv, q, a.M_out, ctx->K, ctx->O_rep, ctx->m_rep, ctx->l_rep, s);
  if (spec) cudaStreamWaitEvent(s, ctx->ev_spec, 0);  // join
  launch_merge(ctx, kv->batch, ctx->merge_src, ctx->merge_n, ctx->O_spec, ctx->m_spec, ctx->l_spec,
               ctx->Bud, ctx->O_rep, ctx->m_rep, ctx->l_rep, ctx->K, out, nullptr, nullptr, s);
  return check_launch(ctx, "prr_decode_step");
}

extern "C" int32_t prr_step_append(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const void* k_new,
                                   const void* v_new, void* summaries, float* out, int32_t sequential,
                                   void* stream) {
  NO_FP8("prr_step_append");
  CHECK_KV("prr_step_append");
  CHECK_PTR(q, "prr_step_append"); CHECK_PTR(k_new, "prr_step_append"); CHECK_PTR(v_new, "prr_step_append");
  CHECK_PTR(summaries, "prr_step_append");
  if (!out) PRR_FAIL(ctx, PRR_E_INVALID, "prr_step_append: null out");
  if (ctx->fused)  // a0 rides in the same launch as a1-a8
    return fused_step(ctx, kv, q, summaries, out, sequential ? 0 : 1, (cudaStream_t)stream, "prr_step_append",
                      k_new, v_new);
  const int r = prr_append(ctx, kv, k_new, v_new, summaries, stream);
  if (r) return r;
  return sequential ? prr_attend(ctx, kv, q, summaries, out, stream)
                    : prr_decode_step(ctx, kv, q, summaries, out, stream);
}

extern "C" int32_t prr_decode_step_host(prr_ctx* ctx, const prr_paged_kv* kv, const void* q_host,
                                        const void* k_new_host, const void* v_new_host, void* summaries,
                                        float* out_host, void* stream) {
  NO_FP8("prr_decode_step_host");
  CHECK_KV("prr_decode_step_host");
  if (!q_host || !k_new_host || !v_new_host || !out_host || !summaries)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_decode_step_host: null argument");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t qb = (size_t)kv->batch * ctx->Hq * ctx->D, kb = (size_t)kv->batch * ctx->Hkv * ctx->D;
  // one host->device copy: the three inputs are packed (at the layout of a full batch: the device
  // pointers st_q / st_k / st_v are fixed offsets) into the pinned staging buffer first.  The call
  // synchronises the stream before it returns, so the buffer is free again on the next call.
  const size_t qfull = (size_t)ctx->maxB * ctx->Hq * ctx->D, kfull = (size_t)ctx->maxB * ctx->Hkv * ctx->D;
  uint16_t* pin = (uint16_t*)ctx->st_pin;
  memcpy(pin, q_host, qb * 2);
  memcpy(pin + qfull, k_new_host, kb * 2);
  memcpy(pin + qfull + kfull, v_new_host, kb * 2);
  const size_t span = kv->batch == ctx->maxB ? qfull + 2 * kfull : 0;
  if (span) {
    PRR_CUDA(ctx, cudaMemcpyAsync(ctx->st_q, pin, span * 2, cudaMemcpyHostToDevice, s));
  } else {  // partial batch: the three parts are not contiguous on the device side
    PRR_CUDA(ctx, cudaMemcpyAsync(ctx->st_q, pin, qb * 2, cudaMemcpyHostToDevice, s));
    PRR_CUDA(ctx, cudaMemcpyAsync(ctx->st_k, pin + qfull, kb * 2, cudaMemcpyHostToDevice, s));
    PRR_CUDA(ctx, cudaMemcpyAsync(ctx->st_v, pin + qfull + kfull, kb * 2, cudaMemcpyHostToDevice, s));
  }
  // Result: a device->host copy command after the kernel costs ~17 us of queueing for 16 KB (measured, DESIGN.md
  // section 9), so a small result is stored by the kernel itself straight into host memory: the caller's buffer when it
  // is pinned and mapped (cudaHostAlloc / torch pin_memory), else a mapped staging buffer copied out after the sync.
  // A large result (batch serving) keeps the copy engine: its stores would hold the reducer warps on PCIe.
  float* out_d = ctx->st_out;
  bool direct = false, staged = false;
  if (qb * sizeof(float) <= HOST_OUT_DIRECT) {
    if (out_host != ctx->out_seen) {
      cudaPointerAttributes pa{};
      ctx->out_seen = out_host; ctx->out_seen_d = nullptr;
      if (cudaPointerGetAttributes(&pa, out_host) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer)
        ctx->out_seen_d = (float*)pa.devicePointer;
      cudaGetLastError();
    }
    if (ctx->out_seen_d) { out_d = ctx->out_seen_d; direct = true; }
    else { out_d = ctx->st_out_hd; staged = true; }
  }
  // A result the kernel stores into host memory is announced the same way: the step's last warp stores a sequence
  // number into a mapped host word (system-scope release after every result); polling it costs ~1 us where
  // cudaStreamSynchronize costs the driver's wake-up.  Later work on `stream` is stream-ordered behind the kernel as usual.
  const bool poll = (direct || staged) && ctx->fused && ctx->done_h;
  uint32_t seq = 0;
  if (poll) { seq = ++ctx->done_seq ? ctx->done_seq : ++ctx->done_seq; ctx->arm_seq = seq; }
  const int r = prr_step_append(ctx, kv, ctx->st_q, ctx->st_k, ctx->st_v, summaries, out_d, 0, stream);
  ctx->arm_seq = 0;
  if (r) return r;
  if (!direct && !staged) PRR_CUDA(ctx, cudaMemcpyAsync(out_host, ctx->st_out, qb * sizeof(float), cudaMemcpyDeviceToHost, s));
  bool seen = false;
  if (poll) {
    const auto t0 = std::chrono::steady_clock::now();
    for (uint32_t it = 0; !(seen = *ctx->done_h == seq); ++it) {
      if ((it & 0xfffu) == 0xfffu) {  // give up polling after 50 ms (a failed launch never stores the word): synchronise instead
        if (std::chrono::steady_clock::now() - t0 > std::chrono::milliseconds(50)) break;
        if (cudaStreamQuery(s) != cudaErrorNotReady) break;
      }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
  }
  if (!seen) PRR_CUDA(ctx, cudaStreamSynchronize(s));
  if (staged) memcpy(out_host, ctx->st_out_h, qb * sizeof(float));
  return PRR_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" int32_t prr_get_sets(prr_ctx* ctx, int32_t layer, int32_t batch, int32_t* A, int32_t* P,
                                int32_t* M, int32_t* counts, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || batch < 1 || batch > ctx->maxB)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_get_sets: layer/batch out of range");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  const size_t r = layer_rows(ctx, layer), n = (size_t)batch * ctx->Hkv;
  if (A) PRR_CUDA(ctx, cudaMemcpyAsync(A, ctx->setA + r * ctx->K, n * ctx->K * 4, cudaMemcpyDeviceToDevice, s));
  if (M) PRR_CUDA(ctx, cudaMemcpyAsync(M, ctx->setM + r * ctx->K, n * ctx->K * 4, cudaMemcpyDeviceToDevice, s));
  if (P && ctx->Bud > 0 && ctx->fused) {
    const size_t np = n * ctx->Bud;
    k_copy_P<<<(unsigned)((np + 255) / 256), 256, 0, s>>>(ctx->Pbuf[0] + r * ctx->Bud, ctx->Pbuf[1] + r * ctx->Bud,
                                                          ctx->parity + layer, 1, P, np, 0);
    ctx->launches++;
  } else if (P && ctx->Bud > 0)
    PRR_CUDA(ctx, cudaMemcpyAsync(P, ctx->P_used + r * ctx->Bud, n * ctx->Bud * 4, cudaMemcpyDeviceToDevice, s));
  if (counts) PRR_CUDA(ctx, cudaMemcpyAsync(counts, ctx->counts + r * 3, n * 3 * 4, cudaMemcpyDeviceToDevice, s));
  return PRR_OK;
}

extern "C" int32_t prr_get_scores(prr_ctx* ctx, int32_t layer, int32_t batch, float* scores, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || batch < 1 || batch > ctx->maxB || !scores)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_get_scores: bad argument");
  const size_t r = layer_rows(ctx, layer), n = (size_t)batch * ctx->Hkv * ctx->MB;
  PRR_CUDA(ctx, cudaMemcpyAsync(scores, ctx->scores + r * ctx->MB, n * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return PRR_OK;
}

extern "C" int32_t prr_get_ema(prr_ctx* ctx, int32_t layer, int32_t seq, double* level, double* trend,
                               int32_t* n_state, double* theta, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (layer < 0 || layer >= ctx->NL || seq < 0 || seq >= ctx->maxB)
    PRR_FAIL(ctx, PRR_E_INVALID, "prr_get_ema: layer/seq out of range");
  cudaStream_t s = (cudaStream_t)stream;
  join_layer(ctx, layer, s);
  const size_t sq = (size_t)layer * ctx->maxB + seq, n = (size_t)ctx->Hkv * ctx->MB;
  if (level) PRR_CUDA(ctx, cudaMemcpyAsync(level, ctx->ema_l + sq * n, n * 8, cudaMemcpyDeviceToDevice, s));
  if (trend) PRR_CUDA(ctx, cudaMemcpyAsync(trend, ctx->ema_v + sq * n, n * 8, cudaMemcpyDeviceToDevice, s));
  if (n_state) PRR_CUDA(ctx, cudaMemcpyAsync(n_state, ctx->n_state + sq * ctx->Hkv, ctx->Hkv * 4, cudaMemcpyDeviceToDevice, s));
  if (theta) {
    PRR_CUDA(ctx, cudaMemcpyAsync(theta, ctx->theta + sq * 3, 24, cudaMemcpyDeviceToHost, s));
    PRR_CUDA(ctx, cudaStreamSynchronize(s));
  }
  return PRR_OK;
}

extern "C" int32_t prr_get_stats(prr_ctx* ctx, int64_t* stats_out, int32_t reset, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  join_updates(ctx, s);
  if (stats_out) PRR_CUDA(ctx, cudaMemcpyAsync(stats_out, ctx->stats, 32, cudaMemcpyDeviceToHost, s));
  if (reset) PRR_CUDA(ctx, cudaMemsetAsync(ctx->stats, 0, 32, s));
  PRR_CUDA(ctx, cudaStreamSynchronize(s));
  return PRR_OK;
}

extern "C" int32_t prr_check(prr_ctx* ctx, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  join_updates(ctx, s);
  uint32_t err[4] = {0, 0, 0, 0};  // ctl[1] error flag ... ctl[4] first wait site that gave up (k_row.cu)
  PRR_CUDA(ctx, cudaMemcpyAsync(err, ctx->ctl + 1, sizeof(err), cudaMemcpyDeviceToHost, s));
  PRR_CUDA(ctx, cudaStreamSynchronize(s));
  if (err[0])
    PRR_FAIL(ctx, PRR_E_STATE, "prr_check: a fused step gave up waiting on a dependency (site %u, CTA %u, warp %u)",
             err[3] & 0xffu, (err[3] >> 8) & 0xfffu, err[3] >> 20);
  return check_launch(ctx, "prr_check");
}

extern "C" int32_t prr_set_option(prr_ctx* ctx, int32_t option, int32_t value) {
  if (!ctx) return PRR_E_INVALID;
  switch (option) {
    case PRR_OPT_PDL: if (value != 0 && value != 1) break; ctx->pdl = value; return PRR_OK;
    case PRR_OPT_CLUSTER: if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 && value != 16) break; ctx->force_cs = value; return PRR_OK;
    case PRR_OPT_CUT: if (value != 0 && value != 1) break; ctx->cut = value; return PRR_OK;
    case PRR_OPT_SUBTILE: if (value != 16 && value != 32 && value != 64) break; ctx->sub_tile = value; ctx->tmaps.clear(); return PRR_OK;
    case PRR_OPT_KERNEL: if (value < 0 || value > 2) break; ctx->kernel = value; ctx->tmaps.clear(); return PRR_OK;
    case PRR_OPT_PACE: if (value < 0 || value > 1000) break; ctx->pace_pct = value; return PRR_OK;
    case PRR_OPT_SUMMARY:
      if (value != PRR_SUMMARY_MEAN && value != PRR_SUMMARY_QUEST) break;
      if (value == PRR_SUMMARY_QUEST && ctx->fused)
        PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_option: the fused kernels score mean summaries only; create the context with "
                 "orchestration PRR_STREAMS to use Quest min/max summaries");
      ctx->summary_kind = value; return PRR_OK;
    default: break;
  }
  PRR_FAIL(ctx, PRR_E_INVALID, "prr_set_option: unknown option %d or bad value %d", option, value);
}

extern "C" int32_t prr_get_option(const prr_ctx* ctx, int32_t option, int32_t* value_out) {
  if (!ctx || !value_out) return PRR_E_INVALID;
  switch (option) {
    case PRR_OPT_PDL: *value_out = ctx->pdl; return PRR_OK;
    case PRR_OPT_CLUSTER: *value_out = ctx->force_cs; return PRR_OK;
    case PRR_OPT_CUT: *value_out = ctx->cut; return PRR_OK;
    case PRR_OPT_SUBTILE: *value_out = ctx->sub_tile; return PRR_OK;
    case PRR_OPT_KERNEL: *value_out = ctx->kernel; return PRR_OK;
    case PRR_OPT_PACE: *value_out = ctx->pace_pct; return PRR_OK;
    case PRR_OPT_SUMMARY: *value_out = ctx->summary_kind; return PRR_OK;
    case PRR_OPT_LAST_KERNEL: *value_out = ctx->last_kernel; return PRR_OK;
    case PRR_OPT_LAST_CLUSTER: *value_out = ctx->last_cs; return PRR_OK;
    case PRR_OPT_LAST_RING: *value_out = ctx->last_nbuf; return PRR_OK;
    case PRR_OPT_LAST_GRID: *value_out = ctx->last_grid; return PRR_OK;
    default: return PRR_E_INVALID;
  }
}

extern "C" int32_t prr_timeline_enable(prr_ctx* ctx, int32_t on) {
  if (!ctx) return PRR_E_INVALID;
  ctx->tl_on = on ? 1 : 0;
  return PRR_OK;
}

extern "C" int32_t prr_timeline_read(prr_ctx* ctx, uint64_t* stamps_host, int32_t max_warps, int32_t* n_warps_out,
                                     void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (!stamps_host || max_warps < 1) PRR_FAIL(ctx, PRR_E_INVALID, "prr_timeline_read: bad argument");
  cudaStream_t s = (cudaStream_t)stream;
  const int n = max_warps < ctx->tl_warps ? max_warps : ctx->tl_warps;
  PRR_CUDA(ctx, cudaStreamSynchronize(s));
  memcpy(stamps_host, ctx->tl, (size_t)n * 16 * sizeof(uint64_t));
  if (n_warps_out) *n_warps_out = n;
  return PRR_OK;
}

extern "C" int32_t prr_timeline_peek(prr_ctx* ctx, uint64_t* stamps_host, int32_t max_warps, int32_t* n_warps_out) {
  if (!ctx) return PRR_E_INVALID;
  if (!stamps_host || max_warps < 1) PRR_FAIL(ctx, PRR_E_INVALID, "prr_timeline_peek: bad argument");
  const int n = max_warps < ctx->tl_warps ? max_warps : ctx->tl_warps;
  memcpy(stamps_host, ctx->tl, (size_t)n * 16 * sizeof(uint64_t));
  if (n_warps_out) *n_warps_out = n;
  return PRR_OK;
}

// ---------------------------------------------------------------------------------------------
extern "C" int32_t prr_graph_begin(prr_ctx* ctx, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  join_updates(ctx, s);  // side work issued before the capture must not be waited on inside it
  PRR_CUDA(ctx, cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
  return PRR_OK;
}

extern "C" int32_t prr_graph_end(prr_ctx* ctx, void* stream, prr_graph** out) {
  if (!ctx || !out) return PRR_E_INVALID;
  cudaStream_t s = (cudaStream_t)stream;
  join_updates(ctx, s);  // every forked branch rejoins the origin stream before the capture ends
  prr_graph* g = new prr_graph();
  cudaError_t e = cudaStreamEndCapture(s, &g->graph);
  if (e == cudaSuccess) e = cudaGraphInstantiate(&g->exec, g->graph, 0);
  if (e == cudaSuccess) e = cudaGraphUpload(g->exec, s);  // the first launch does not pay for the upload
  if (e != cudaSuccess) {
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;
    cudaGetLastError();
    PRR_FAIL(ctx, PRR_E_CUDA, "prr_graph_end: %s", cudaGetErrorString(e));
  }
  *out = g;
  return PRR_OK;
}

extern "C" int32_t prr_graph_launch(prr_graph* g, void* stream) {
  if (!g || !g->exec) return PRR_E_INVALID;
  return cudaGraphLaunch(g->exec, (cudaStream_t)stream) == cudaSuccess ? PRR_OK : PRR_E_CUDA;
}

extern "C" int32_t prr_graph_destroy(prr_graph* g) {
  if (!g) return PRR_E_INVALID;
  if (g->exec) cudaGraphExecDestroy(g->exec);
  if (g->graph) cudaGraphDestroy(g->graph);
  delete g;
  return PRR_OK;
}
