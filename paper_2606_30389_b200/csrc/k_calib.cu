// Per-prompt EMA calibration: Eq. 4 score-weighted hit rate over the prefill
// trajectory for the 80-point (alpha, beta, gamma) grid, Eq. 5 first argmax.  Three launches:
//   k_calib_truth  grid (T, Hkv): A_phi = top-K of row phi -> bitmask + denominator sum_A IS
//   k_calib_sim    grid (80, Hkv): the sequential Eq. 2-3 simulation of one theta on one KV head
//   k_calib_final  1 CTA: H(theta) in head order, first maximiser, seeds the layer's EMA state
// Readings Q5/Q8: |P_phi| = min(Bud, #stateful); the stateful blocks at row phi are
// those valid at row phi-1; rows without state or with a non-positive denominator are skipped.
#include "prr_dev.cuh"
#include "prr_internal.h"

namespace prr {

constexpr int CAL_NT = 256;
constexpr int N_THETA = 80;

__device__ __forceinline__ double block_sum_f64(double x, double* wtmp) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) x += __shfl_xor_sync(FULL, x, off);
  __syncthreads();
  if (lane == 0) wtmp[warp] = x;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int w = 0; w < CAL_NT / 32; ++w) t += wtmp[w];
  return t;
}

struct CalSmem {
  unsigned long long* scan;  // 40 x u64 (also used as 8 doubles by block_sum_f64)
  uint32_t* keys;
  uint32_t* mask;
  uint32_t* hist;
  uint32_t* ctl;
};
__device__ __forceinline__ CalSmem cal_carve(unsigned char* base, int N, int words) {
  CalSmem s;
  s.scan = reinterpret_cast<unsigned long long*>(base);
  s.keys = reinterpret_cast<uint32_t*>(base + 40 * 8);
  s.mask = s.keys + N;
  s.hist = s.mask + words;
  s.ctl = s.hist + 256;
  return s;
}
static size_t cal_smem_bytes(int N) { return 40 * 8 + ((size_t)N + (N + 31) / 32 + 256 + 8) * 4; }

__global__ void __launch_bounds__(CAL_NT)
k_calib_truth(const float* __restrict__ IS, const int32_t* __restrict__ n_valid, int T, int N, int K,
              uint32_t* __restrict__ maskA, double* __restrict__ den) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, phi = blockIdx.x, h = blockIdx.y;
  const int words = (N + 31) / 32;
  CalSmem s = cal_carve(smem_raw, N, words);
  const int n = n_valid ? min(N, n_valid[phi]) : N;
  const float* row = IS + ((size_t)h * T + phi) * N;
  for (int w = tid; w < words; w += CAL_NT) s.mask[w] = 0;
  for (int i = tid; i < n; i += CAL_NT) s.keys[i] = score_key(row[i]);
  __syncthreads();
  const int k = min(K, n);
  if (k > 0) {
    uint32_t Tk;
    int need;
    radix_select<CAL_NT>(s.keys, n, k, s.hist, s.ctl, Tk, need);
    ordered_select<CAL_NT>(s.keys, n, Tk, need, nullptr, s.mask, s.scan);
  }
  __syncthreads();
  double loc = 0.0;
  uint32_t* out = maskA + ((size_t)h * T + phi) * words;
  for (int w = tid; w < words; w += CAL_NT) {
    uint32_t m = s.mask[w];
    out[w] = m;
    while (m) {
      const int bit = __ffs(m) - 1;
      m &= m - 1;
      loc += (double)row[w * 32 + bit];
    }
  }
  const double d = block_sum_f64(loc, reinterpret_cast<double*>(s.scan));
  if (tid == 0) den[(size_t)h * T + phi] = d;
}

__device__ __forceinline__ void theta_of(int ti, double& alpha, double& beta, double& gamma) {
  alpha = __ddiv_rn((double)(2 * (ti / 20 + 1)), 10.0);
  beta = __ddiv_rn((double)((ti / 4) % 5 + 1), 10.0);
  gamma = __ddiv_rn((double)(ti % 4), 4.0);
}

__global__ void __launch_bounds__(CAL_NT)
k_calib_sim(const float* __restrict__ IS, const int32_t* __restrict__ n_valid, int T, int N, int Bud,
            int Hkv, const uint32_t* __restrict__ maskA, const double* __restrict__ den,
            double* __restrict__ state, double* __restrict__ acc_out, int32_t* __restrict__ cnt_out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, ti = blockIdx.x, h = blockIdx.y;
  const int words = (N + 31) / 32;
  CalSmem s = cal_carve(smem_raw, N, words);
  double alpha, beta, gamma;
  theta_of(ti, alpha, beta, gamma);
  const double oma = __dsub_rn(1.0, alpha), omb = __dsub_rn(1.0, beta);
  double* L = state + ((size_t)ti * Hkv + h) * 2 * N;
  double* V = L + N;
  double acc = 0.0;
  int cnt = 0;
  int n_st = 0;
  for (int phi = 0; phi < T; ++phi) {
    const int n = n_valid ? min(N, n_valid[phi]) : N;
    const float* row = IS + ((size_t)h * T + phi) * N;
    if (n_st > 0) {
      for (int w = tid; w < words; w += CAL_NT) s.mask[w] = 0;
      for (int i = tid; i < n_st; i += CAL_NT)
        s.keys[i] = score_key(f64_to_score(__dadd_rn(L[i], __dmul_rn(gamma, V[i]))));
      __syncthreads();
      if (min(Bud, n_st) > 0) {
        uint32_t Tk;
        int need;
        radix_select<CAL_NT>(s.keys, n_st, min(Bud, n_st), s.hist, s.ctl, Tk, need);
        ordered_select<CAL_NT>(s.keys, n_st, Tk, need, nullptr, s.mask, s.scan);
      }
      __syncthreads();
      const uint32_t* mA = maskA + ((size_t)h * T + phi) * words;
      double loc = 0.0;
      for (int w = tid; w < words; w += CAL_NT) {
        uint32_t m = s.mask[w] & mA[w];
        while (m) {
          const int bit = __ffs(m) - 1;
          m &= m - 1;
          loc += (double)row[w * 32 + bit];
        }
      }
      const double num = block_sum_f64(loc, reinterpret_cast<double*>(s.scan));
      const double d = den[(size_t)h * T + phi];
      if (d > 0.0) {  // Eq. 4 summand; accumulated in row order
        acc = __dadd_rn(acc, __ddiv_rn(num, d));
        ++cnt;
      }
    }
    for (int i = tid; i < n; i += CAL_NT) {
      const double x = (double)row[i];
      if (i < n_st) {
        const double lo = L[i], vo = V[i];
        V[i] = __dadd_rn(__dmul_rn(beta, __dsub_rn(x, lo)), __dmul_rn(omb, vo));
        L[i] = __dadd_rn(__dmul_rn(alpha, x), __dmul_rn(oma, lo));
      } else {
        L[i] = x;
        V[i] = 0.0;
      }
    }
    n_st = max(n_st, n);
    __syncthreads();
  }
  if (tid == 0) {
    acc_out[ti * Hkv + h] = acc;
    cnt_out[ti * Hkv + h] = cnt;
  }
}

__global__ void __launch_bounds__(128)
k_calib_final(const double* __restrict__ acc, const int32_t* __restrict__ cnt, int Hkv, int N,
              const int32_t* __restrict__ n_valid, int T, const double* __restrict__ state,
              double* __restrict__ H_out,
              int32_t* __restrict__ best_out, double* __restrict__ theta, double* __restrict__ ema_l,
              double* __restrict__ ema_v, int32_t* __restrict__ n_state, int MB) {
  __shared__ double Hs[N_THETA];
  __shared__ int best_s;
  const int tid = threadIdx.x;
  const int n_last = n_valid ? min(N, n_valid[T - 1]) : N;
  if (tid < N_THETA) {
    double total = 0.0;
    long long count = 0;
    for (int h = 0; h < Hkv; ++h) {
      total = __dadd_rn(total, acc[tid * Hkv + h]);
      count += cnt[tid * Hkv + h];
    }
    const double H = count ? __ddiv_rn(total, (double)count) : 0.0;
    Hs[tid] = H;
    H_out[tid] = H;
  }
  __syncthreads();
  if (tid == 0) {
    int best = 0;
    for (int t = 1; t < N_THETA; ++t)
      if (Hs[t] > Hs[best]) best = t;  // first maximiser (Eq. 5)
    best_s = best;
    *best_out = best;
    double a, b, g;
    theta_of(best, a, b, g);
    theta[0] = a;
    theta[1] = b;
    theta[2] = g;
  }
  __syncthreads();
  const int best = best_s;
  for (int h = 0; h < Hkv; ++h) {
    const double* L = state + ((size_t)best * Hkv + h) * 2 * N;
    for (int i = tid; i < n_last; i += blockDim.x) {
      ema_l[(size_t)h * MB + i] = L[i];
      ema_v[(size_t)h * MB + i] = L[N + i];
    }
    if (tid == 0) n_state[h] = n_last;
  }
}

static bool ensure(prr_ctx* c, void** p, size_t* have, size_t need_bytes) {
  if (*have >= need_bytes) return true;
  if (*p) cudaFree(*p);
  *p = nullptr;
  *have = 0;
  if (cudaMalloc(p, need_bytes) != cudaSuccess) { c->err = "prr_calibrate: out of device memory"; return false; }
  *have = need_bytes;
  return true;
}

int launch_calibrate(prr_ctx* c, int layer, int seq, const float* IS, int T, int N,
                     const int32_t* n_valid, cudaStream_t s) {
  const int words = (N + 31) / 32;
  size_t b1 = c->cal_state_elems * sizeof(double), b2 = c->cal_mask_words * 4, b3 = c->cal_den_elems * 8;
  if (!ensure(c, (void**)&c->cal_state, &b1, (size_t)N_THETA * c->Hkv * 2 * N * sizeof(double))) return PRR_E_NOMEM;
  if (!ensure(c, (void**)&c->cal_mask, &b2, (size_t)c->Hkv * T * words * 4)) return PRR_E_NOMEM;
  if (!ensure(c, (void**)&c->cal_den, &b3, (size_t)c->Hkv * T * 8)) return PRR_E_NOMEM;
  c->cal_state_elems = b1 / sizeof(double);
  c->cal_mask_words = b2 / 4;
  c->cal_den_elems = b3 / 8;

  const size_t smem = cal_smem_bytes(N);
  if (smem > 48 * 1024) {
    cudaFuncSetAttribute((const void*)k_calib_truth, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute((const void*)k_calib_sim, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  double* acc = c->cal_acc;                                        // [80*Hkv]
  int32_t* cnt = reinterpret_cast<int32_t*>(acc + N_THETA * c->Hkv);  // [80*Hkv]
  double* H = acc + 2 * N_THETA * c->Hkv;                          // [80]
  int32_t* best = reinterpret_cast<int32_t*>(H + N_THETA);
  k_calib_truth<<<dim3(T, c->Hkv), CAL_NT, smem, s>>>(IS, n_valid, T, N, c->K, c->cal_mask, c->cal_den);
  k_calib_sim<<<dim3(N_THETA, c->Hkv), CAL_NT, smem, s>>>(IS, n_valid, T, N, c->Bud, c->Hkv, c->cal_mask,
                                                          c->cal_den, c->cal_state, acc, cnt);
  const size_t sq = (size_t)layer * c->maxB + seq;
  k_calib_final<<<1, 128, 0, s>>>(acc, cnt, c->Hkv, N, n_valid, T, c->cal_state, H, best,
                                  c->theta + sq * 3, c->ema_l + sq * c->Hkv * c->MB,
                                  c->ema_v + sq * c->Hkv * c->MB, c->n_state + sq * c->Hkv, c->MB);
  c->launches += 3;
  return PRR_OK;
}

}  // namespace prr
