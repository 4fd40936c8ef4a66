// prr_attend_blocks_static — sparse attention over given block lists (a4 + a7, Eq. 6-8)
// for callers that may not allocate: code under stream capture, tight serving loops, harnesses that forbid
// cudaMalloc.  The per-block partial states (m, l, O) that the split-KV attention of this library keeps
// between its two launches normally live in buffers the prr_ctx allocated; here they live in ONE file-scope
// device array of PRR_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit.
//
//   * the array's name is a host-side stand-in in host code, not a device address: its address is resolved
//     with cudaGetSymbolAddress, once per device, with that device current, and only that pointer is
//     ever handed to a kernel;
//   * every call shares the array and it keeps the last call's contents.  Nothing in it has to start at
//     zero: every slot that is read was written by the same call (slots whose list entry is -1 are neither
//     written nor read);
//   * calls that overlap on the GPU (two streams, two host threads, two contexts on one device) RACE on
//     it: order them on one stream or with events.
#include <math_constants.h>

#include <cstdio>
#include <mutex>

#include "prr_dev.cuh"
#include "prr_internal.h"

// 8 MiB: batch * n_q_heads * width * (head_dim + 2) floats, e.g. batch 1 x 32 heads x 496 blocks at d = 128
static __device__ __align__(256) float g_static_scratch[PRR_STATIC_SCRATCH_BYTES / 4];

namespace prr {
namespace {

constexpr float LOG2E_S = 1.4426950408889634f;

// Variant of k_merge (k_attn.cu) whose partial states come from the static scratch: one CTA per (query
// head, sequence) folds the states of the listed blocks in list order (holes of -1 skipped) with the
// log-sum-exp rescaling of Eq. 6-8, O unnormalised, one division at the end.  Same three passes and the
// same reduction shapes as k_merge, so the two agree to the last bit on the same states.
template <int D>
__global__ void __launch_bounds__(4 * D)
k_merge_static(const int32_t* __restrict__ list, int width, const float* __restrict__ O_part,
               const float* __restrict__ m_part, const float* __restrict__ l_part, float* __restrict__ out,
               float* __restrict__ m_out, float* __restrict__ l_out, int Hq, int Hkv, int G) {
  constexpr int NT = 4 * D;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* ws = reinterpret_cast<float*>(smem_raw);             // [width] weights
  int32_t* cs = reinterpret_cast<int32_t*>(ws + width);       // [width] slots, compacted
  __shared__ float red[4 * D];
  __shared__ float wred[NT / 32];
  __shared__ float bc[2];
  __shared__ int n_sh;
  const int hq = blockIdx.x, b = blockIdx.y, h = hq / G;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int32_t* src = list + ((size_t)b * Hkv + h) * width;
  const size_t hb = (size_t)b * Hq + hq;
  if (warp == 0) {  // slots with a block, in list order
    int n = 0;
    for (int j0 = 0; j0 < width; j0 += 32) {
      const int j = j0 + lane;
      const bool on = j < width && src[j] >= 0;
      const uint32_t bal = __ballot_sync(FULL, on);
      if (on) cs[n + __popc(bal & ((1u << lane) - 1u))] = j;
      n += __popc(bal);
    }
    if (lane == 0) n_sh = n;
  }
  __syncthreads();
  const int n = n_sh;
  float mx = -CUDART_INF_F;
  for (int e = tid; e < n; e += NT) {
    const float me = m_part[hb * width + cs[e]];
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
  float lsum = 0.f;
  for (int e = tid; e < n; e += NT) {
    const float me = ws[e];
    const float w = me == -CUDART_INF_F ? 0.f : ex2((me - m_all) * LOG2E_S);
    ws[e] = w;
    lsum = fmaf(w, l_part[hb * width + cs[e]], lsum);
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
  const int grp = tid / D, c = tid - grp * D;
  float acc = 0.f;
#pragma unroll 4
  for (int e = grp; e < n; e += 4) acc = fmaf(ws[e], O_part[(hb * width + cs[e]) * D + c], acc);
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

// Device address of the scratch array on the CURRENT device, resolved once per device.
constexpr int MAX_DEV = 64;
std::mutex g_mu;
float* g_scratch_ptr[MAX_DEV] = {};

cudaError_t scratch_address(float** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_scratch_ptr[dev]) {
    float* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_scratch);  // (not &g_static_scratch: that is a host address)
    if (e != cudaSuccess) return e;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

int fail(prr_ctx* c, int code, const char* msg) {
  if (c) c->err = msg;
  return code;
}

}  // namespace
}  // namespace prr

using namespace prr;

extern "C" int64_t prr_static_scratch_bytes(void) { return (int64_t)PRR_STATIC_SCRATCH_BYTES; }

extern "C" int32_t prr_attend_blocks_static(prr_ctx* ctx, const prr_paged_kv* kv, const void* q, const int32_t* blocks,
                                            int32_t width, float* out, float* m_out, float* l_out, void* stream) {
  if (!ctx) return PRR_E_INVALID;
  if (!kv || !kv->k_pages || !kv->v_pages || !kv->block_table || !kv->seq_lens)
    return fail(ctx, PRR_E_INVALID, "prr_attend_blocks_static: null paged-KV field");
  if (kv->batch < 1 || kv->batch > ctx->maxB) return fail(ctx, PRR_E_INVALID, "prr_attend_blocks_static: batch out of range");
  if (!q || !blocks || !out) return fail(ctx, PRR_E_INVALID, "prr_attend_blocks_static: null argument");
  if (width < 1 || width > 1024) return fail(ctx, PRR_E_INVALID, "prr_attend_blocks_static: width must be 1 .. 1024");
  if (kv->layer < 0 || kv->layer >= ctx->NL) return fail(ctx, PRR_E_INVALID, "prr_attend_blocks_static: layer out of range");
  if (ctx->lay.kv_dtype == PRR_FP8_E4M3 && (!ctx->kscale[kv->layer] || !ctx->vscale[kv->layer]))
    return fail(ctx, PRR_E_STATE, "prr_attend_blocks_static: fp8 KV: call prr_set_kv_scales first");
  if (ctx->bs > 128) return fail(ctx, PRR_E_UNSUPPORTED, "prr_attend_blocks_static: blocks of 256 tokens run on the fused step only");
  const size_t slots = (size_t)kv->batch * ctx->Hq * (size_t)width;
  const size_t need = slots * (size_t)(ctx->D + 2) * sizeof(float);
  if (need > (size_t)PRR_STATIC_SCRATCH_BYTES) {
    char b[256];
    snprintf(b, sizeof(b), "prr_attend_blocks_static: batch %d x %d query heads x width %d x (d + 2) floats = %zu bytes "
             "exceeds the static scratch of %d bytes", kv->batch, ctx->Hq, width, need, (int)PRR_STATIC_SCRATCH_BYTES);
    return fail(ctx, PRR_E_UNSUPPORTED, b);
  }
  float* base = nullptr;
  cudaError_t e = scratch_address(&base);
  if (e != cudaSuccess) {
    cudaGetLastError();
    char b[256];
    snprintf(b, sizeof(b), "prr_attend_blocks_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    return fail(ctx, PRR_E_CUDA, b);
  }
  float* O = base;                         // [batch, n_q_heads, width, d]
  float* m = base + slots * ctx->D;        // [batch, n_q_heads, width]
  float* l = m + slots;                    // [batch, n_q_heads, width]
  cudaStream_t s = (cudaStream_t)stream;
  launch_partial(ctx, kv, q, blocks, width, O, m, l, s);
  const size_t smem = (size_t)width * 8;
  dim3 grid(ctx->Hq, kv->batch);
  if (ctx->D == 128)
    k_merge_static<128><<<grid, 512, smem, s>>>(blocks, width, O, m, l, out, m_out, l_out, ctx->Hq, ctx->Hkv, ctx->G);
  else
    k_merge_static<64><<<grid, 256, smem, s>>>(blocks, width, O, m, l, out, m_out, l_out, ctx->Hq, ctx->Hkv, ctx->G);
  ctx->launches++;
  e = cudaPeekAtLastError();
  if (e != cudaSuccess) {
    cudaGetLastError();
    char b[256];
    snprintf(b, sizeof(b), "prr_attend_blocks_static: %s", cudaGetErrorString(e));
    return fail(ctx, PRR_E_CUDA, b);
  }
  return PRR_OK;
}
