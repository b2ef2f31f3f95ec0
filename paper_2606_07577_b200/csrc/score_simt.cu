// SIMT scoring kernels: score pass 1 (row LSE of Eq.1's softmax) and pass 2 (Eq.6 column sums).
// Used for fp32 inputs (CFG1, 1e-5 tolerance: no tensor-core rounding allowed) and for bf16 shapes the
// tcgen05 path does not cover (head_dim != 128).  One warp per query row (pass 1) / per key (pass 2).
#include <math.h>

#include "common.cuh"

namespace omnimem {

template <typename T> struct Vec16;
template <> struct Vec16<float> {
  static constexpr int N = 4;
  __device__ static __forceinline__ void load(const float* p, float* o) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(p));
    o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
  }
};
template <> struct Vec16<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ static __forceinline__ void load(const __nv_bfloat16* p, float* o) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      o[2 * i] = __uint_as_float(w[i] << 16);
      o[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  }
};
__device__ __forceinline__ float to_float(float x) { return x; }
__device__ __forceinline__ float to_float(__nv_bfloat16 x) { return __bfloat162float(x); }

template <typename T>
__device__ __forceinline__ float dot_row(const float* __restrict__ sx, const T* __restrict__ gy, int D) {
  float acc = 0.f;
  for (int d = 0; d < D; d += Vec16<T>::N) {
    float y[Vec16<T>::N];
    Vec16<T>::load(gy + d, y);
#pragma unroll
    for (int e = 0; e < Vec16<T>::N; ++e) acc = fmaf(sx[d + e], y[e], acc);
  }
  return acc;
}

// ---- pass 1: lse[l,j,i] = log sum_{k visible} exp(c <q_i, k_k>)   (softmax of P:54 Eq.1; needed by Eq.6) ----
template <typename T, bool kEntropy>
__global__ void __launch_bounds__(128) lse_simt_kernel(StepParams p, const T* __restrict__ cacheK,
                                                       const T* __restrict__ chunkK, const T* __restrict__ Q,
                                                       float* __restrict__ lse, float* __restrict__ rowH) {
  extern __shared__ float sq[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long row = (long long)blockIdx.x * 4 + warp;
  if (row >= (long long)p.L * p.Hq * p.Nn) return;
  const int i = (int)(row % p.Nn);
  const int j = (int)((row / p.Nn) % p.Hq);
  const int l = (int)(row / ((long long)p.Nn * p.Hq));
  if (layer_skips_scoring(p, l)) return;
  const int h = j / p.G, D = p.D;
  const T* q = Q + row * D;
  float* myq = sq + warp * D;
  for (int d = lane; d < D; d += 32) myq[d] = to_float(q[d]);
  __syncwarp();
  const int Nc = p.n[l];
  const int nvis = p.causal ? Nc + i + 1 : Nc + p.Nn;
  const T* kc = cacheK + (long long)(l * p.Hkv + h) * p.cache_cap * D;
  const T* kn = chunkK + (long long)(l * p.Hkv + h) * p.Nn * D;
  float m = -INFINITY, Z = 0.f, W = 0.f;
  for (int k = lane; k < nvis; k += 32) {
    const T* kr = k < Nc ? kc + (long long)k * D : kn + (long long)(k - Nc) * D;
    const float z = p.scale * dot_row<T>(myq, kr, D);
    if (z > m) {
      const float r = expf(m - z);
      Z = Z * r + 1.f;
      if (kEntropy) W = W * r + z;
      m = z;
    } else {
      const float e = expf(z - m);
      Z += e;
      if (kEntropy) W = fmaf(e, z, W);
    }
  }
  float mm = m;
#pragma unroll
  for (int o = 16; o; o >>= 1) mm = fmaxf(mm, __shfl_xor_sync(0xffffffffu, mm, o));
  const float r = (m == -INFINITY) ? 0.f : expf(m - mm);
  Z *= r;
  W *= r;
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    Z += __shfl_xor_sync(0xffffffffu, Z, o);
    W += __shfl_xor_sync(0xffffffffu, W, o);
  }
  if (lane == 0) {
    const float v = mm + logf(Z);
    lse[row] = v;
    if (kEntropy) rowH[row] = v - W / Z;  // -sum p ln p = lse - sum p z
  }
}

// ---- pass 2: a[l,h,k] = sum_g sum_{i visible} exp(c <q_i, k_k> - lse[l,hG+g,i])   (Eq.6, R5) ----
template <typename T>
__global__ void __launch_bounds__(128) colsum_simt_kernel(StepParams p, const T* __restrict__ cacheK,
                                                          const T* __restrict__ chunkK, const T* __restrict__ Q,
                                                          const float* __restrict__ lse, float* __restrict__ a_v,
                                                          float* __restrict__ a_a) {
  extern __shared__ float sk[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int slots = p.cache_cap + p.Nn;  // logical key slots per (l,h): cache rows by capacity, then chunk rows
  const long long item = (long long)blockIdx.x * 4 + warp;
  if (item >= (long long)p.L * p.Hkv * slots) return;
  const int kk = (int)(item % slots);
  const int h = (int)((item / slots) % p.Hkv);
  const int l = (int)(item / ((long long)slots * p.Hkv));
  if (layer_skips_scoring(p, l)) return;
  const int D = p.D, n_v = p.n_v[l], n = p.n[l];
  int m, t, t_chunk = -1;
  const T* kr;
  if (kk < p.cache_cap) {
    if (kk >= n) return;
    kr = cacheK + ((long long)(l * p.Hkv + h) * p.cache_cap + kk) * D;
    cache_row_to_seg(n_v, kk, m, t);
  } else {
    t_chunk = kk - p.cache_cap;
    kr = chunkK + ((long long)(l * p.Hkv + h) * p.Nn + t_chunk) * D;
    chunk_row_to_seg(p, n_v, n, t_chunk, m, t);
  }
  float* myk = sk + warp * D;
  for (int d = lane; d < D; d += 32) myk[d] = to_float(kr[d]);
  __syncwarp();
  float acc = 0.f;
  const int rows = p.G * p.Nn;
  for (int rr = lane; rr < rows; rr += 32) {
    const int g = rr / p.Nn, i = rr % p.Nn;
    if (p.causal && t_chunk > i) continue;
    const long long qrow = (long long)(l * p.Hq + h * p.G + g) * p.Nn + i;
    const float z = p.scale * dot_row<T>(myk, Q + qrow * D, D);
    acc += expf(z - lse[qrow]);
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) {
    float* out = m == 0 ? a_v + (long long)(l * p.Hkv + h) * p.seg_cap_v : a_a + (long long)(l * p.Hkv + h) * p.seg_cap_a;
    out[t] = acc;
  }
}

// ---- Eq.1: Y[l,j,i,:] = sum_k exp(c <q_i, k_k> - lse[l,j,i]) v_k, given the row LSE of pass 1 ----
// One block per query row: 128 keys at a time, thread t takes key t's weight, then thread d accumulates output column d
// over the 128 weights (coalesced value reads).  fp32 throughout; serves fp32 inputs and head_dim != 128.
__device__ __forceinline__ void store_out(float* p, float v) { *p = v; }
__device__ __forceinline__ void store_out(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

template <typename T>
__global__ void __launch_bounds__(128) attend_simt_kernel(StepParams p, const T* __restrict__ cacheK,
                                                          const T* __restrict__ cacheV, const T* __restrict__ chunkK,
                                                          const T* __restrict__ chunkV, const T* __restrict__ Q,
                                                          const float* __restrict__ lse, T* __restrict__ Y) {
  extern __shared__ float sm_att[];
  const int i = blockIdx.x, j = blockIdx.y, l = blockIdx.z, t = threadIdx.x;
  const int h = j / p.G, D = p.D;
  float* sq = sm_att;         // [D]
  float* sp = sm_att + D;     // [128]
  const long long row = ((long long)l * p.Hq + j) * p.Nn + i;
  for (int d = t; d < D; d += 128) sq[d] = to_float(Q[row * D + d]);
  __syncthreads();
  const int Nc = p.n[l];
  const int nvis = p.causal ? Nc + i + 1 : Nc + p.Nn;
  const long long lh = (long long)l * p.Hkv + h;
  const T* kc = cacheK + lh * p.cache_cap * D;
  const T* vc = cacheV + lh * p.cache_cap * D;
  const T* kn = chunkK + lh * p.Nn * D;
  const T* vn = chunkV + lh * p.Nn * D;
  const float row_lse = lse[row];
  float acc = 0.f;
  for (int k0 = 0; k0 < nvis; k0 += 128) {
    const int k = k0 + t;
    float w = 0.f;
    if (k < nvis) {
      const T* kr = k < Nc ? kc + (long long)k * D : kn + (long long)(k - Nc) * D;
      w = expf(p.scale * dot_row<T>(sq, kr, D) - row_lse);
    }
    sp[t] = w;
    __syncthreads();
    const int cnt = min(128, nvis - k0);
    for (int d = t; d < D; d += 128)
      for (int u = 0; u < cnt; ++u) {
        const int kk = k0 + u;
        const T* vr = kk < Nc ? vc + (long long)kk * D : vn + (long long)(kk - Nc) * D;
        acc = fmaf(sp[u], to_float(vr[d]), acc);
      }
    __syncthreads();
  }
  for (int d = t; d < D; d += 128) store_out(Y + row * D + d, acc);
}

// ---- Eq.6 below fp32's range (R31) ---------------------------------------------------------------------
// Both column-sum kernels add fp32 weights: a weight below 2^-126 is flushed, so a key that NO query attends to comes
// out as 0 (or as a sum that lost most of its terms) although Eq.8 raises it to lambda = 0.02, which maps 1e-80 to 0.025:
// the ranking among unattended keys lives in that range.  Keys whose fp32 sum is below 2^-100 (at most G Nq lost
// terms of < 2^-126 each cannot move a larger sum by 1e-3) are therefore recomputed here in the log domain,
//     la = log2 sum_{g,i visible} 2^(c2 <q_i, k> - lse2_i)      (per-lane running maximum, merged across the warp),
// and finalize takes psi = 2^(lambda la) (1 - s) for them.  Weights below 2^-1074 are dropped: fp64, the oracle's type,
// ends there, and psi jumps from 3e-7 to 0 at that point in the oracle as well.  One warp looks at 32 consecutive key
// slots and works through the flagged ones; with ordinary logits nothing is flagged and the kernel is one load per key.
constexpr float kTinyImportance = 7.888609052210118e-31f;   // 2^-100

template <typename T>
__global__ void __launch_bounds__(128) colsum_rescue_kernel(StepParams p, const T* __restrict__ cacheK,
                                                            const T* __restrict__ chunkK, const T* __restrict__ Q,
                                                            const float* __restrict__ lse_arr, int lse_stride, float lse_coef,
                                                            float* __restrict__ a_v, float* __restrict__ a_a,
                                                            float* __restrict__ la_v, float* __restrict__ la_a) {
  extern __shared__ float sk[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int slots = p.cache_cap + p.Nn;               // logical key slots per (l,h): cache rows by capacity, then chunk rows
  const int groups = (slots + 31) / 32;
  const long long item = (long long)blockIdx.x * 4 + warp;
  if (item >= (long long)p.L * p.Hkv * groups) return;
  const int grp = (int)(item % groups);
  const int h = (int)((item / groups) % p.Hkv);
  const int l = (int)(item / ((long long)groups * p.Hkv));
  if (layer_skips_scoring(p, l)) return;
  const int D = p.D, n_v = p.n_v[l], n = p.n[l];
  const long long lh = (long long)l * p.Hkv + h;
  auto locate = [&](int kk, int& m, int& t, int& t_chunk) -> bool {   // slot -> (modality, segment index); false = no key there
    t_chunk = -1;
    if (kk >= slots) return false;
    if (kk < p.cache_cap) {
      if (kk >= n) return false;
      cache_row_to_seg(n_v, kk, m, t);
    } else {
      t_chunk = kk - p.cache_cap;
      chunk_row_to_seg(p, n_v, n, t_chunk, m, t);
    }
    return true;
  };
  int m, t, t_chunk;
  const bool valid = locate(grp * 32 + lane, m, t, t_chunk);
  float av = 1.f;
  if (valid) av = (m == 0 ? a_v + lh * p.seg_cap_v : a_a + lh * p.seg_cap_a)[t];
  unsigned todo = __ballot_sync(0xffffffffu, valid && !(av >= kTinyImportance));
  float* myk = sk + warp * D;
  const int rows = p.G * p.Nn;
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    locate(grp * 32 + src, m, t, t_chunk);
    const T* kr = t_chunk < 0 ? cacheK + (lh * p.cache_cap + (grp * 32 + src)) * D : chunkK + (lh * p.Nn + t_chunk) * D;
    __syncwarp();
    for (int d = lane; d < D; d += 32) myk[d] = to_float(kr[d]);
    __syncwarp();
    float mx = -INFINITY, z = 0.f;
    for (int rr = lane; rr < rows; rr += 32) {
      const int g = rr / p.Nn, i = rr % p.Nn;
      if (p.causal && t_chunk > i) continue;
      const long long qh = (long long)l * p.Hq + h * p.G + g;
      const float x = fmaf(p.scale_log2e, dot_row<T>(myk, Q + (qh * p.Nn + i) * D, D), lse_coef * lse_arr[qh * lse_stride + i]);
      if (x < -1074.f) continue;   // below the smallest fp64 number: such a weight is 0 in the oracle's arithmetic too
      if (x > mx) { z = z * exp2f(mx - x) + 1.f; mx = x; } else z += exp2f(x - mx);
    }
    float M = mx;
#pragma unroll
    for (int o = 16; o; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    z = mx == -INFINITY ? 0.f : z * exp2f(mx - M);
#pragma unroll
    for (int o = 16; o; o >>= 1) z += __shfl_xor_sync(0xffffffffu, z, o);
    if (lane == 0) {
      const float la = z > 0.f ? M + log2f(z) : -INFINITY;
      (m == 0 ? la_v + lh * p.seg_cap_v : la_a + lh * p.seg_cap_a)[t] = la;
      (m == 0 ? a_v + lh * p.seg_cap_v : a_a + lh * p.seg_cap_a)[t] = exp2f(la);   // what fp32 can hold of it (usually 0)
    }
  }
}

template <typename T>
static cudaError_t lse_simt_t(const StepParams& p, const StepBuffers& b, cudaStream_t st) {
  const long long rows = (long long)p.L * p.Hq * p.Nn;
  if (rows == 0) return cudaSuccess;
  const unsigned grid = (unsigned)((rows + 3) / 4);
  const size_t smem = 4 * p.D * sizeof(float);
  if (b.row_entropy)
    lse_simt_kernel<T, true><<<grid, 128, smem, st>>>(p, (const T*)b.cacheK, (const T*)b.chunkK, (const T*)b.Q, b.lse,
                                                      b.row_entropy);
  else
    lse_simt_kernel<T, false><<<grid, 128, smem, st>>>(p, (const T*)b.cacheK, (const T*)b.chunkK, (const T*)b.Q, b.lse,
                                                       nullptr);
  return cudaGetLastError();
}

cudaError_t launch_lse_simt(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st,
                            int* launches) {
  if ((long long)p.L * p.Hq * p.Nn == 0) return cudaSuccess;
  ++*launches;
  return ctx->cfg.dtype == OMNIMEM_FP32 ? lse_simt_t<float>(p, b, st) : lse_simt_t<__nv_bfloat16>(p, b, st);
}

// pass 1 (LSE, natural log, into lse_nat) then the weighted value sum
cudaError_t launch_attend_simt(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, void* y, float* lse_nat,
                               cudaStream_t st, int* launches) {
  if ((long long)p.L * p.Hq * p.Nn == 0) return cudaSuccess;
  StepBuffers b2 = b;
  b2.lse = lse_nat;
  b2.row_entropy = nullptr;
  cudaError_t e = launch_lse_simt(ctx, p, b2, st, launches);
  if (e != cudaSuccess) return e;
  const dim3 grid((unsigned)p.Nn, (unsigned)p.Hq, (unsigned)p.L);
  const size_t smem = (size_t)(p.D + 128) * sizeof(float);
  ++*launches;
  if (ctx->cfg.dtype == OMNIMEM_FP32)
    attend_simt_kernel<float><<<grid, 128, smem, st>>>(p, (const float*)b.cacheK, (const float*)b.cacheV, (const float*)b.chunkK,
                                                       (const float*)b.chunkV, (const float*)b.Q, lse_nat, (float*)y);
  else
    attend_simt_kernel<__nv_bfloat16><<<grid, 128, smem, st>>>(p, (const __nv_bfloat16*)b.cacheK, (const __nv_bfloat16*)b.cacheV,
                                                               (const __nv_bfloat16*)b.chunkK, (const __nv_bfloat16*)b.chunkV,
                                                               (const __nv_bfloat16*)b.Q, lse_nat, (__nv_bfloat16*)y);
  return cudaGetLastError();
}

cudaError_t launch_colsum_simt(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st,
                               int* launches) {
  const long long items = (long long)p.L * p.Hkv * (p.cache_cap + p.Nn);
  if (items == 0) return cudaSuccess;
  const unsigned grid = (unsigned)((items + 3) / 4);
  const size_t smem = 4 * p.D * sizeof(float);
  ++*launches;
  if (ctx->cfg.dtype == OMNIMEM_FP32)
    colsum_simt_kernel<float><<<grid, 128, smem, st>>>(p, (const float*)b.cacheK, (const float*)b.chunkK,
                                                       (const float*)b.Q, b.lse, b.a_v, b.a_a);
  else
    colsum_simt_kernel<__nv_bfloat16><<<grid, 128, smem, st>>>(p, (const __nv_bfloat16*)b.cacheK,
                                                               (const __nv_bfloat16*)b.chunkK,
                                                               (const __nv_bfloat16*)b.Q, b.lse, b.a_v, b.a_a);
  return cudaGetLastError();
}

}  // namespace omnimem

namespace omnimem {

// SIMT path: per-key recompute against the natural-log LSE.  tcgen05 path: launch_colsum_rescue_tc (score_tc.cu).
cudaError_t launch_colsum_rescue(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st,
                                 int* launches) {
  if (p.Nn == 0) return cudaSuccess;     // no queries: a = 0 everywhere by definition, psi = 0^lambda (1 - s)
  // tensor-core path: the flagged 256-key items go through the scoring kernel once more (bounded by one more pass 2); the
  // per-key kernel below costs a flagged key as much as the SIMT pass 2 does, which is the right bound only on the SIMT path
  if (ctx->use_tc) return launch_colsum_rescue_tc(ctx, p, b, st, launches);
  const int groups = (p.cache_cap + p.Nn + 31) / 32;
  const long long items = (long long)p.L * p.Hkv * groups;
  const unsigned grid = (unsigned)((items + 3) / 4);
  const size_t smem = 4 * p.D * sizeof(float);
  const float* lse_arr = b.lse;          // the natural-log LSE of the SIMT passes
  const int stride = p.Nn;
  const float coef = -1.4426950408889634f;
  ++*launches;
  if (ctx->cfg.dtype == OMNIMEM_FP32)
    colsum_rescue_kernel<float><<<grid, 128, smem, st>>>(p, (const float*)b.cacheK, (const float*)b.chunkK, (const float*)b.Q,
                                                         lse_arr, stride, coef, b.a_v, b.a_a, b.la_v, b.la_a);
  else
    colsum_rescue_kernel<__nv_bfloat16><<<grid, 128, smem, st>>>(p, (const __nv_bfloat16*)b.cacheK, (const __nv_bfloat16*)b.chunkK,
                                                                 (const __nv_bfloat16*)b.Q, lse_arr, stride, coef, b.a_v, b.a_a,
                                                                 b.la_v, b.la_a);
  return cudaGetLastError();
}

}  // namespace omnimem
