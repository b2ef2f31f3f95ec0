// Bandwidth / latency kernels of the step: adjacent cosine (Eq.7), finalize (Eq.8 psi + Eq.9-10/13 partial
// statistics), statistics + budgets (Eq.9-14), segmented radix top-M (Eq.4-5), gather-compaction.
#include <math.h>

#include "common.cuh"

namespace omnimem {

// ------------------------------------------------------------------------------------------------------------
// Eq.7 (value rows per P:103, R8): cosn[t] = cos(x_t, x_{t+sigma}) inside the modality's appended sequence.
// s_t is assembled from cosn[t] and cosn[t-sigma] in finalize.  kTPR threads (16 B each) cover one row.
// ------------------------------------------------------------------------------------------------------------
// 16 bytes of a row and of its partner: dot += <x, y>, nx += <x, x>, ny += <y, y> in fp32.
template <typename T> struct Vec16;
template <> struct Vec16<float> {
  __device__ static __forceinline__ void acc(const uint4& x, const uint4& y, float& dot, float& nx, float& ny) {
    const float xs[4] = {__uint_as_float(x.x), __uint_as_float(x.y), __uint_as_float(x.z), __uint_as_float(x.w)};
    const float ys[4] = {__uint_as_float(y.x), __uint_as_float(y.y), __uint_as_float(y.z), __uint_as_float(y.w)};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      dot = fmaf(xs[e], ys[e], dot);
      nx = fmaf(xs[e], xs[e], nx);
      ny = fmaf(ys[e], ys[e], ny);
    }
  }
};
template <> struct Vec16<__nv_bfloat16> {
  // mixed-precision FMA (bf16 x bf16 + fp32, exact products): no unpacking of the bf16 pairs
  __device__ static __forceinline__ void fma_pair(float& d0, float& d1, uint32_t a, uint32_t b) {
    asm("{\n\t.reg .b16 al, ah, bl, bh;\n\tmov.b32 {al, ah}, %2;\n\tmov.b32 {bl, bh}, %3;\n\t"
        "fma.rn.f32.bf16 %0, al, bl, %0;\n\tfma.rn.f32.bf16 %1, ah, bh, %1;\n\t}" : "+f"(d0), "+f"(d1) : "r"(a), "r"(b));
  }
  __device__ static __forceinline__ void acc(const uint4& x, const uint4& y, float& dot, float& nx, float& ny) {
    const uint32_t xs[4] = {x.x, x.y, x.z, x.w}, ys[4] = {y.x, y.y, y.z, y.w};
    float d1 = 0.f, nx1 = 0.f, ny1 = 0.f;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      fma_pair(dot, d1, xs[e], ys[e]);
      fma_pair(nx, nx1, xs[e], xs[e]);
      fma_pair(ny, ny1, ys[e], ys[e]);
    }
    dot += d1; nx += nx1; ny += ny1;
  }
};

// kTPR = 4 threads cover one row, kVec 16-byte vectors each (vector j of the row goes to thread j % 4, so a warp's load
// instruction touches 8 rows x 64 contiguous bytes).  One block works on kUnroll * 64 consecutive items of one (layer, KV
// head) at a time; every thread first issues all of its 2 * kUnroll * kVec loads (row t and its partner t + sigma, which
// comes out of L1 / L2), then reduces: ~25 instructions per 16 bytes instead of ~115 (the first version was
// instruction-bound: ncu, profiles/).
// Round 3: a block alternates a load phase and a reduce phase, so what hides one block's latency is the OTHER resident
// blocks, not more loads per thread.  With kUnroll = 2 the bf16 kernel took 92 registers = 2 blocks per SM (ncu: 24 % warps
// active, 56 % of the HBM copy peak); kUnroll = 1 under __launch_bounds__(256, 4) takes 56 registers = 4 blocks per SM with
// the same bytes in flight per SM: config 2 0.196 -> 0.120 ms (5.35 TB/s, 82 % of the measured copy peak), config 3
// 0.907 -> 0.573 ms (88 %).  (3 blocks of the kUnroll = 2 form: 0.149 / 0.693 ms.)
// Items are numbered DENSELY over the rows that exist (K_v visual, then K_a audio: device counts), and a fixed number of
// blocks per (layer, KV head) strides over them: sized by capacity, 43 % of the blocks of config 2 had no row to read and
// their launch overhead alone was a quarter of the kernel's time.
template <typename T, int kVec, int kUnroll>
__global__ void __launch_bounds__(256, kVec * kUnroll <= 4 ? 4 : 3) cosine_kernel(StepParams p, const T* __restrict__ cacheX,
                                                     const T* __restrict__ chunkX, float* __restrict__ cosn) {
  constexpr int kTPR = 4, kRows = 256 / kTPR;
  const int items = p.seg_cap_v + p.seg_cap_a;
  const int lh = blockIdx.y, l = lh / p.Hkv;
  if (layer_skips_scoring(p, l)) return;
  const int sub = threadIdx.x % kTPR;
  const int n_v = p.n_v[l], n = p.n[l];
  const int Kv = seg_len(p, n_v, n, 0), Ka = seg_len(p, n_v, n, 1);
  const uint4* cbase = reinterpret_cast<const uint4*>(cacheX + (long long)lh * p.cache_cap * p.D) + sub;
  const uint4* kbase = reinterpret_cast<const uint4*>(chunkX + (long long)lh * p.Nn * p.D) + sub;
  const int row_vecs = kVec * kTPR;
  for (int d0 = blockIdx.x * (kUnroll * kRows); d0 < Kv + Ka; d0 += gridDim.x * (kUnroll * kRows)) {
    uint4 xv[kUnroll][kVec], yv[kUnroll][kVec];
    bool active[kUnroll];
    int out[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const int d = d0 + u * kRows + threadIdx.x / kTPR;      // dense item: visual rows, then audio rows
      const int m = d < Kv ? 0 : 1;
      const int t = m == 0 ? d : d - Kv;
      const int sg = m == 0 ? p.stride_v : p.stride_a;
      out[u] = m == 0 ? t : p.seg_cap_v + t;
      active[u] = d < Kv + Ka && t + sg < (m == 0 ? Kv : Ka);
      if (active[u]) {
        bool cx, cy;
        const int rx = seg_row(p, n_v, n, m, t, cx), ry = seg_row(p, n_v, n, m, t + sg, cy);
        const uint4* x = (cx ? kbase : cbase) + (long long)rx * row_vecs;
        const uint4* y = (cy ? kbase : cbase) + (long long)ry * row_vecs;
#pragma unroll
        for (int i = 0; i < kVec; ++i) { xv[u][i] = __ldg(x + i * kTPR); yv[u][i] = __ldg(y + i * kTPR); }
      }
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      float dot = 0.f, nx = 0.f, ny = 0.f;
      if (active[u]) {
#pragma unroll
        for (int i = 0; i < kVec; ++i) Vec16<T>::acc(xv[u][i], yv[u][i], dot, nx, ny);
      }
#pragma unroll
      for (int o = kTPR / 2; o; o >>= 1) {
        dot += __shfl_xor_sync(0xffffffffu, dot, o);
        nx += __shfl_xor_sync(0xffffffffu, nx, o);
        ny += __shfl_xor_sync(0xffffffffu, ny, o);
      }
      if (active[u] && sub == 0) cosn[(long long)lh * items + out[u]] = dot / fmaxf(sqrtf(nx) * sqrtf(ny), 1e-8f);  // R12
    }
  }
}

// Eq.7 in the paper's first form: the vectors are the layer's hidden states H_k, one row of d_model elements
// per token and layer ([L, cache_cap, d_model] / [L, Nn, d_model]; R30).  One warp per item streams row t and row
// t + sigma in 512-byte steps (4 steps in flight), so the sweep is one pass over H at HBM speed; the cosine is written
// to every KV head's slot of cosn, finalize then runs unchanged.
template <typename T>
__global__ void __launch_bounds__(256) cosine_hidden_kernel(StepParams p, const T* __restrict__ cacheH,
                                                            const T* __restrict__ chunkH, float* __restrict__ cosn) {
  const int items = p.seg_cap_v + p.seg_cap_a;
  const int l = blockIdx.y;
  if (layer_skips_scoring(p, l)) return;
  const int lane = threadIdx.x & 31;
  const int it = blockIdx.x * 8 + (threadIdx.x >> 5);
  if (it >= items) return;
  const int n_v = p.n_v[l], n = p.n[l];
  const int m = it < p.seg_cap_v ? 0 : 1;
  const int t = m == 0 ? it : it - p.seg_cap_v;
  const int sg = m == 0 ? p.stride_v : p.stride_a;
  if (t + sg >= seg_len(p, n_v, n, m)) return;
  bool cx, cy;
  const int rx = seg_row(p, n_v, n, m, t, cx), ry = seg_row(p, n_v, n, m, t + sg, cy);
  const int row_vecs = p.d_model * (int)sizeof(T) / 16;
  const uint4* x = reinterpret_cast<const uint4*>(cx ? chunkH + ((long long)l * p.Nn + rx) * p.d_model
                                                     : cacheH + ((long long)l * p.cache_cap + rx) * p.d_model);
  const uint4* y = reinterpret_cast<const uint4*>(cy ? chunkH + ((long long)l * p.Nn + ry) * p.d_model
                                                     : cacheH + ((long long)l * p.cache_cap + ry) * p.d_model);
  float dot = 0.f, nx = 0.f, ny = 0.f;
  constexpr int kU = 4;
  for (int v0 = lane; v0 < row_vecs; v0 += 32 * kU) {
    uint4 xv[kU], yv[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u)
      if (v0 + 32 * u < row_vecs) { xv[u] = __ldg(x + v0 + 32 * u); yv[u] = __ldg(y + v0 + 32 * u); }
#pragma unroll
    for (int u = 0; u < kU; ++u)
      if (v0 + 32 * u < row_vecs) Vec16<T>::acc(xv[u], yv[u], dot, nx, ny);
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    dot += __shfl_xor_sync(0xffffffffu, dot, o);
    nx += __shfl_xor_sync(0xffffffffu, nx, o);
    ny += __shfl_xor_sync(0xffffffffu, ny, o);
  }
  const float c = dot / fmaxf(sqrtf(nx) * sqrtf(ny), 1e-8f);  // R12
  for (int h = lane; h < p.Hkv; h += 32) cosn[((long long)l * p.Hkv + h) * items + it] = c;
}

cudaError_t launch_cosine(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st,
                          int* launches) {
  const int items = p.seg_cap_v + p.seg_cap_a;
  if (ctx->cfg.sim_source == 2) {
    const dim3 grid((unsigned)((items + 7) / 8), (unsigned)p.L);
    ++*launches;
    if (ctx->cfg.dtype == OMNIMEM_FP32)
      cosine_hidden_kernel<float><<<grid, 256, 0, st>>>(p, (const float*)b.cacheH, (const float*)b.chunkH, b.cosn);
    else
      cosine_hidden_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(p, (const __nv_bfloat16*)b.cacheH,
                                                                 (const __nv_bfloat16*)b.chunkH, b.cosn);
    return cudaGetLastError();
  }
  const void* cx = ctx->cfg.sim_source == 0 ? b.cacheV : b.cacheK;
  const void* kx = ctx->cfg.sim_source == 0 ? b.chunkV : b.chunkK;
  const int row_bytes = p.D * (ctx->cfg.dtype == OMNIMEM_FP32 ? 4 : 2);
  const int vec = row_bytes / 64;                      // 16-byte vectors per thread (4 threads per row): 2, 4 or 8
  const int unroll = 1;
  const int rows_per_block = unroll * 64;
  // a fixed number of blocks per (layer, KV head) strides over the rows that exist (device counts): just under 8 full
  // waves of the resident blocks per SM (4; 3 for 512-byte fp32 rows), so that no wave is left mostly empty and no block
  // finds nothing to do
  const int lh_count = p.L * p.Hkv;
  int per_lh = ctx->sm_count * (vec == 8 ? 3 : 4) * 8 / lh_count;
  const int need = (items + rows_per_block - 1) / rows_per_block;
  if (per_lh > need) per_lh = need;
  if (per_lh < 1) per_lh = 1;
  const dim3 grid((unsigned)per_lh, (unsigned)lh_count);
  ++*launches;
#define OMNIMEM_COS(T, V, U) cosine_kernel<T, V, U><<<grid, 256, 0, st>>>(p, (const T*)cx, (const T*)kx, b.cosn)
  if (ctx->cfg.dtype == OMNIMEM_FP32) {
    if (vec == 4) OMNIMEM_COS(float, 4, 1); else OMNIMEM_COS(float, 8, 1);
  } else {
    if (vec == 2) OMNIMEM_COS(__nv_bfloat16, 2, 1); else OMNIMEM_COS(__nv_bfloat16, 4, 1);
  }
#undef OMNIMEM_COS
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Finalize: s_t (Eq.7 mean over existing neighbours, clamp, R10/R12), psi = a^lambda (1-s) (Eq.8), and per-block
// partial sums of A_t = sum_h a, A_t ln A_t and s for the AVBA statistics (Eq.9-10, 13; H = ln S - sum A ln A / S).
// ------------------------------------------------------------------------------------------------------------
// a^lambda with the log-domain value for the keys below fp32's range (R31; colsum_rescue_kernel wrote la for exactly the
// keys with a < 2^-100); C pow semantics at the ends: x^0 = 1, 0^lambda = 0 (R13)
__device__ __forceinline__ float pow_importance(float a, float la, float lambda) {
  if (a >= 7.888609052210118e-31f) return powf(a, lambda);
  return lambda == 0.f ? 1.f : exp2f(lambda * la);
}

__global__ void __launch_bounds__(256) finalize_kernel(StepParams p, const float* __restrict__ a_v,
                                                       const float* __restrict__ a_a, const float* __restrict__ la_v,
                                                       const float* __restrict__ la_a, const float* __restrict__ cosn,
                                                       float* __restrict__ s_v, float* __restrict__ s_a,
                                                       float* __restrict__ psi_v, float* __restrict__ psi_a,
                                                       double* __restrict__ partials, int nblk) {
  const int l = blockIdx.z, m = blockIdx.y, t = blockIdx.x * 256 + threadIdx.x;
  const int n_v = p.n_v[l], n = p.n[l];
  const int Km = seg_len(p, n_v, n, m);
  const int cap = m == 0 ? p.seg_cap_v : p.seg_cap_a;
  const int sg = m == 0 ? p.stride_v : p.stride_a;
  const int items = p.seg_cap_v + p.seg_cap_a;
  const bool skip = layer_skips_scoring(p, l);
  double v0 = 0.0, v1 = 0.0, v2 = 0.0;
  if (t < Km && !skip) {
    float A = 0.f, ssum = 0.f, la_max = -INFINITY;
    for (int h = 0; h < p.Hkv; ++h) {
      const long long lh = (long long)l * p.Hkv + h;
      const float* cs = cosn + lh * items + (m == 0 ? 0 : p.seg_cap_v);
      float sum = 0.f;
      int cnt = 0;
      if (t + sg < Km) { sum += cs[t]; ++cnt; }
      if (t - sg >= 0) { sum += cs[t - sg]; ++cnt; }
      float s = cnt == 2 ? 0.5f * sum : sum;  // cnt == 0 -> 0 (R10)
      s = fminf(1.f, fmaxf(-1.f, s));
      const float a = (m == 0 ? a_v : a_a)[lh * cap + t];
      const float la = a >= 7.888609052210118e-31f ? 0.f : (p.Nn > 0 ? (m == 0 ? la_v : la_a)[lh * cap + t] : -INFINITY);
      (m == 0 ? s_v : s_a)[lh * cap + t] = s;
      if (!p.shared_heads) (m == 0 ? psi_v : psi_a)[lh * cap + t] = pow_importance(a, la, p.lambda) * (1.f - s);
      else if (a < 7.888609052210118e-31f) la_max = fmaxf(la_max, la);
      A += a;
      ssum += s;
    }
    if (p.shared_heads) {  // R29: one score per token and layer, written to every head's row (identical index sets)
      float LA = la_max;   // log2 of the sum over heads, needed only when even the sum is below fp32's range
      if (A < 7.888609052210118e-31f && la_max > -INFINITY) {
        float zs = 0.f;
        for (int h = 0; h < p.Hkv; ++h) zs += exp2f((m == 0 ? la_v : la_a)[((long long)l * p.Hkv + h) * cap + t] - la_max);
        LA = la_max + log2f(zs);
      }
      const float psi = pow_importance(A, LA, p.lambda) * (1.f - ssum / (float)p.Hkv);
      for (int h = 0; h < p.Hkv; ++h) (m == 0 ? psi_v : psi_a)[((long long)l * p.Hkv + h) * cap + t] = psi;
    }
    v0 = (double)A;
    v1 = A > 0.f ? (double)A * log((double)A) : 0.0;
    v2 = (double)ssum;
  }
  __shared__ double red[3][8];
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    v0 += __shfl_xor_sync(0xffffffffu, v0, o);
    v1 += __shfl_xor_sync(0xffffffffu, v1, o);
    v2 += __shfl_xor_sync(0xffffffffu, v2, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) { red[0][warp] = v0; red[1][warp] = v1; red[2][warp] = v2; }
  __syncthreads();
  if (threadIdx.x < 3) {
    double acc = 0.0;
    for (int w = 0; w < 8; ++w) acc += red[threadIdx.x][w];
    partials[(((long long)l * 2 + m) * nblk + blockIdx.x) * 3 + threadIdx.x] = acc;
  }
}

// stats[l] = {Hn_v, Hn_a, sbar_v, sbar_a, C_v, C_a, Hn_all, sbar_all}; one warp per layer, fixed summation order.
__global__ void __launch_bounds__(32) stats_kernel(StepParams p, const double* __restrict__ partials, int nblk,
                                                   double* __restrict__ stats) {
  const int l = blockIdx.x, lane = threadIdx.x;
  double S[2], Tl[2], Ss[2];
  for (int m = 0; m < 2; ++m) {
    double v0 = 0.0, v1 = 0.0, v2 = 0.0;
    const double* pp = partials + ((long long)l * 2 + m) * nblk * 3;
    for (int b = lane; b < nblk; b += 32) { v0 += pp[b * 3]; v1 += pp[b * 3 + 1]; v2 += pp[b * 3 + 2]; }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      v0 += __shfl_xor_sync(0xffffffffu, v0, o);
      v1 += __shfl_xor_sync(0xffffffffu, v1, o);
      v2 += __shfl_xor_sync(0xffffffffu, v2, o);
    }
    S[m] = v0; Tl[m] = v1; Ss[m] = v2;
  }
  if (lane == 0) {
    const int n_v = p.n_v[l], n = p.n[l];
    const int K[2] = {seg_len(p, n_v, n, 0), seg_len(p, n_v, n, 1)};
    double Hn[2], sbar[2];
    for (int m = 0; m < 2; ++m) {
      double H = S[m] > 0.0 ? log(S[m]) - Tl[m] / S[m] : 0.0;
      H = H < 0.0 ? 0.0 : H;
      Hn[m] = (K[m] > 1 && S[m] > 0.0) ? fmin(1.0, H / log((double)K[m])) : 0.0;  // R15
      sbar[m] = K[m] > 0 ? Ss[m] / ((double)K[m] * p.Hkv) : 0.0;                    // R17
    }
    const double Sall = S[0] + S[1], Tall = Tl[0] + Tl[1];
    const int Kall = K[0] + K[1];
    double Hall = Sall > 0.0 ? log(Sall) - Tall / Sall : 0.0;
    Hall = Hall < 0.0 ? 0.0 : Hall;
    double* st = stats + (long long)l * 8;
    st[0] = Hn[0]; st[1] = Hn[1]; st[2] = sbar[0]; st[3] = sbar[1];
    st[4] = Hn[0] * (1.0 - sbar[0]);  // Eq.9
    st[5] = Hn[1] * (1.0 - sbar[1]);  // Eq.10
    st[6] = (Kall > 1 && Sall > 0.0) ? fmin(1.0, Hall / log((double)Kall)) : 0.0;  // Eq.13, R18
    st[7] = Kall > 0 ? (Ss[0] + Ss[1]) / ((double)Kall * p.Hkv) : 0.0;
  }
}

cudaError_t launch_finalize(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st,
                            int* launches) {
  const int nblk = ctx->fin_blocks;
  dim3 grid(nblk, 2, p.L);
  finalize_kernel<<<grid, 256, 0, st>>>(p, b.a_v, b.a_a, b.la_v, b.la_a, b.cosn, b.s_v, b.s_a, b.psi_v, b.psi_a, b.partials, nblk);
  stats_kernel<<<p.L, 32, 0, st>>>(p, b.partials, nblk, b.stats);
  *launches += 2;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Budgets.  Eq.13-14 layer totals (only if layer_budget == nullptr; R19, R20) then Eq.11-12 modality split (R22).
// ------------------------------------------------------------------------------------------------------------
struct AllocParams {
  double ratio_r, temperature;
  long long total_budget, budget_min, budget_max;
};

// Eq.14 with the range [B_min, B_max] of P:137 (R20) is the bounded proportional split
//     b_l = clip(kappa pi_l, B_min, B_max),   kappa such that sum_l b_l = total          ("water-filling").
// f(kappa) = sum_l clip(kappa pi_l, lo, hi) is continuous, non-decreasing and piecewise linear with breakpoints lo / pi_l
// and hi / pi_l.  Thread t evaluates f at breakpoint t (2L of them); the crossing f = total lies between the largest
// breakpoint with f <= total and the smallest with f >= total; between two neighbouring breakpoints the set of layers
// strictly inside the range is constant, so there kappa = (total - mass of the clamped layers) / (pi of the free ones).
// Integerisation is by largest remainder, computed as a RANK: layer l gets one of the `left` spare units iff fewer than
// `left` eligible layers have a larger fractional part (equal parts: the lower layer first) -- no sequential hand-out.
__device__ __forceinline__ double clip_share(double kappa, double pi, double lo, double hi) {
  if (!(pi > 0.0)) return lo;                 // a layer whose softmax weight underflowed sits at the lower bound
  const double v = kappa * pi;
  return v < lo ? lo : (v > hi ? hi : v);
}

__global__ void __launch_bounds__(128) allocate_kernel(StepParams p, AllocParams ap, const double* __restrict__ stats,
                                                       const int32_t* __restrict__ layer_budget, int32_t* __restrict__ M_v,
                                                       int32_t* __restrict__ M_a, int32_t* __restrict__ layer_budget_out) {
  extern __shared__ double sm_alloc[];
  const int L = p.L, tid = threadIdx.x, nthr = blockDim.x;
  double* pi = sm_alloc;               // [L]   softmax over layers
  double* bl = pi + L;                 // [L]   real-valued share
  double* kap = bl + L;                // [2L]  breakpoints
  double* fk = kap + 2 * L;            // [2L]  f at the breakpoints
  int* B = (int*)(fk + 2 * L);         // [L]
  __shared__ double sh_kmid, sh_rem, sh_pfree;
  __shared__ long long sh_left;
  __shared__ int sh_mode;              // 0 = solve, 1 = every layer at B_max, 2 = every layer at B_min
  if (layer_budget != nullptr) {
    for (int l = tid; l < L; l += nthr) B[l] = layer_budget[l];
  } else {
    const bool clamp = ap.budget_max > 0;
    const double lo = clamp ? (double)ap.budget_min : 0.0, hi = clamp ? (double)ap.budget_max : INFINITY;
    const double total = (double)ap.total_budget;
    if (tid == 0) {                      // Eq.13-14: pi = Softmax_l(C^(l) / T), fixed summation order
      double mx = -INFINITY, Z = 0.0;
      for (int l = 0; l < L; ++l) {
        pi[l] = stats[l * 8 + 6] * (1.0 - stats[l * 8 + 7]) / ap.temperature;
        mx = fmax(mx, pi[l]);
      }
      for (int l = 0; l < L; ++l) Z += (pi[l] = exp(pi[l] - mx));
      for (int l = 0; l < L; ++l) pi[l] /= Z;
      sh_mode = (clamp && total >= hi * L) ? 1 : ((clamp && total <= lo * L) ? 2 : 0);
    }
    __syncthreads();
    if (sh_mode != 0) {                  // the range makes the total unreachable: the nearer bound everywhere
      for (int l = tid; l < L; l += nthr) B[l] = (int)(sh_mode == 1 ? ap.budget_max : ap.budget_min);
    } else {
      for (int t = tid; t < 2 * L; t += nthr) {
        const double pl = pi[t < L ? t : t - L];
        const double k = pl > 0.0 ? (t < L ? lo : hi) / pl : INFINITY;
        double f = 0.0;
        for (int l = 0; l < L; ++l) f += clip_share(k, pi[l], lo, hi);
        kap[t] = k;
        fk[t] = f;
      }
      __syncthreads();
      if (tid == 0) {
        double kA = 0.0, kB = INFINITY;    // f(0) = L lo < total < L hi = f(inf)
        for (int t = 0; t < 2 * L; ++t) {
          if (fk[t] <= total && kap[t] > kA && kap[t] < INFINITY) kA = kap[t];
          if (fk[t] >= total && kap[t] < kB) kB = kap[t];
        }
        const double kmid = kB < INFINITY ? 0.5 * (kA + kB) : 2.0 * kA + 1.0;
        double rem = total, pfree = 0.0;
        for (int l = 0; l < L; ++l) {
          const double v = clip_share(kmid, pi[l], lo, hi);
          if (v <= lo || v >= hi) rem -= v; else pfree += pi[l];
        }
        sh_kmid = kmid; sh_rem = rem; sh_pfree = pfree;
      }
      __syncthreads();
      for (int l = tid; l < L; l += nthr) {
        const double v = clip_share(sh_kmid, pi[l], lo, hi);
        bl[l] = (v <= lo || v >= hi) ? v : sh_rem * pi[l] / sh_pfree;
        B[l] = (int)floor(bl[l]);
      }
      __syncthreads();
      if (tid == 0) {
        long long sum = 0;
        for (int l = 0; l < L; ++l) sum += B[l];
        sh_left = ap.total_budget - sum;
      }
      __syncthreads();
      for (int l = tid; l < L; l += nthr) {
        const double fl = floor(bl[l]), fr = bl[l] - fl;
        bool plus = false;
        if (fl + 1.0 <= hi) {
          long long rank = 0;
          for (int j = 0; j < L; ++j) {
            const double fj = floor(bl[j]), rj = bl[j] - fj;
            if (fj + 1.0 <= hi && (rj > fr || (rj == fr && j < l))) ++rank;
          }
          plus = rank < sh_left;
        }
        kap[l] = plus ? 1.0 : 0.0;       // applied after everyone has read bl / B
      }
      __syncthreads();
      for (int l = tid; l < L; l += nthr) B[l] += (int)kap[l];
    }
  }
  __syncthreads();
  for (int l = tid; l < L; l += nthr) {
    // a per-layer total above the cache capacity cannot be stored: it is clamped, not rejected (the budgets are device
    // data, nothing on the host sees them; include/omnimem.h "Budgets")
    const int Bl = B[l] < 0 ? 0 : (B[l] > p.cache_cap ? p.cache_cap : B[l]);
    if (layer_budget_out) layer_budget_out[l] = Bl;
    if (M_v == nullptr) continue;   // calibration: only the per-layer totals are wanted
    const int n_v = p.n_v[l], n = p.n[l];
    const int Kv = seg_len(p, n_v, n, 0), Ka = seg_len(p, n_v, n, 1);
    if (Kv + Ka <= Bl) { M_v[l] = Kv; M_a[l] = Ka; continue; }
    const double Cv = stats[l * 8 + 4], Ca = stats[l * 8 + 5];
    const double den = ap.ratio_r * Cv + Ca;
    const double wv = den > 0.0 ? ap.ratio_r * Cv / den : ap.ratio_r / (ap.ratio_r + 1.0);  // Eq.11
    long long mv = (long long)floor(wv * (double)Bl + 0.5);
    const long long lo = Bl - Ka > 0 ? Bl - Ka : 0, hi = Kv < Bl ? Kv : Bl;
    mv = mv < lo ? lo : (mv > hi ? hi : mv);
    M_v[l] = (int)mv;
    M_a[l] = (int)(Bl - mv);
  }
}

cudaError_t launch_allocate(const omnimem_ctx* ctx, const StepParams& p, const double* stats,
                            const int32_t* layer_budget, int64_t total_budget, int32_t* M_v, int32_t* M_a,
                            int32_t* layer_budget_out, cudaStream_t st, int* launches) {
  AllocParams ap{(double)ctx->cfg.ratio_r, (double)ctx->cfg.temperature, (long long)total_budget,
                 (long long)ctx->cfg.budget_min, (long long)ctx->cfg.budget_max};
  const size_t smem = (size_t)p.L * (6 * sizeof(double) + sizeof(int));
  allocate_kernel<<<1, 128, smem, st>>>(p, ap, stats, layer_budget, M_v, M_a, layer_budget_out);
  ++*launches;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Offline calibration of the per-layer totals ("determined offline ... on a small calibration set", R28):
// acc[l][0..8) += stats[l][0..8) per calibration chunk, acc[L][0] counts the chunks; the budgets are Eq.13-14 on the
// arithmetic means of the two layer measures (normalised entropy, mean similarity).
// ------------------------------------------------------------------------------------------------------------
__global__ void calib_accumulate_kernel(int L, const double* __restrict__ stats, double* __restrict__ acc) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < L * 8) acc[i] += stats[i];
  if (i == 0) acc[L * 8] += 1.0;
}
__global__ void calib_mean_kernel(int L, const double* __restrict__ acc, double* __restrict__ mean) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const double cnt = acc[L * 8];
  if (i < L * 8) mean[i] = cnt > 0.0 ? acc[i] / cnt : 0.0;
}
cudaError_t launch_calib_accumulate(int L, const double* stats, double* acc, cudaStream_t st, int* launches) {
  calib_accumulate_kernel<<<(L * 8 + 127) / 128, 128, 0, st>>>(L, stats, acc);
  ++*launches;
  return cudaGetLastError();
}
cudaError_t launch_calib_mean(int L, const double* acc, double* mean, cudaStream_t st, int* launches) {
  calib_mean_kernel<<<(L * 8 + 127) / 128, 128, 0, st>>>(L, acc, mean);
  ++*launches;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Select (Eq.4-5): per (layer, KV head, modality) the M largest psi, ties -> lowest index, emitted ascending.
// One CTA per segment.  MSB-first radix select on the order-preserving uint image of the fp32 score
// (4 passes x 8 bits, shared-memory histogram with warp-aggregated atomics via match.any), then one ordered
// sweep: rank = #greater before t + min(#equal before t, need), from warp ballots + a scan of warp totals.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t order_key(float x) {
  uint32_t u = __float_as_uint(x);
  if (u == 0x80000000u) u = 0u;  // -0 == +0
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

constexpr int kSelThreads = 1024;

template <bool kSmem>
__global__ void __launch_bounds__(kSelThreads) select_kernel(StepParams p, const float* __restrict__ psi_v,
                                                             const float* __restrict__ psi_a,
                                                             const int32_t* __restrict__ M_v,
                                                             const int32_t* __restrict__ M_a, int32_t* __restrict__ idx_v,
                                                             int32_t* __restrict__ idx_a) {
  extern __shared__ uint32_t skeys[];
  __shared__ uint32_t hist[256];
  __shared__ uint32_t warp_tot[32];
  __shared__ uint32_t warp_off[32];
  __shared__ uint32_t sh_digit, sh_need, sh_chunk_tot;
  const int seg = blockIdx.x;
  const int m = seg & 1, h = (seg >> 1) % p.Hkv, l = (seg >> 1) / p.Hkv;
  const int K = seg_len(p, p.n_v[l], p.n[l], m);
  int Mv_c, Ma_c;
  clamp_budgets(p, p.n_v[l], p.n[l], M_v[l], M_a[l], Mv_c, Ma_c);
  const int M = m == 0 ? Mv_c : Ma_c;
  const long long lh = (long long)l * p.Hkv + h;
  const float* psi = m == 0 ? psi_v + lh * p.seg_cap_v : psi_a + lh * p.seg_cap_a;
  int32_t* out = (m == 0 ? idx_v : idx_a) + lh * p.cache_cap;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (M <= 0) return;
  if (M >= K) {  // nothing to evict in this segment: identity
    for (int t = tid; t < K; t += kSelThreads) out[t] = t;
    return;
  }
  if (kSmem) {
    for (int t = tid; t < K; t += kSelThreads) skeys[t] = order_key(psi[t]);
    __syncthreads();
  }
  auto key = [&](int t) -> uint32_t { return kSmem ? skeys[t] : order_key(__ldg(psi + t)); };
  const int Kpad = (K + kSelThreads - 1) / kSelThreads * kSelThreads;
  uint32_t prefix = 0u, mask = 0u, need = (uint32_t)M;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = 24 - 8 * pass;
    if (tid < 256) hist[tid] = 0u;
    __syncthreads();
    for (int t = tid; t < Kpad; t += kSelThreads) {
      uint32_t d = 256u;  // sentinel: not a candidate
      if (t < K) {
        const uint32_t u = key(t);
        if ((u & mask) == prefix) d = (u >> shift) & 255u;
      }
      const uint32_t peers = __match_any_sync(0xffffffffu, d);
      if (d < 256u && lane == (__ffs(peers) - 1)) atomicAdd(&hist[d], (uint32_t)__popc(peers));
    }
    __syncthreads();
    if (warp == 0) {  // lane i owns bins 255-8i .. 248-8i (descending); find the bin holding the need-th largest
      uint32_t c = 0u;
#pragma unroll
      for (int b = 0; b < 8; ++b) c += hist[255 - 8 * lane - b];
      uint32_t incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      const uint32_t excl = incl - c;
      if (excl < need && need <= incl) {
        uint32_t run = excl;
        for (int b = 0; b < 8; ++b) {
          const int bin = 255 - 8 * lane - b;
          const uint32_t cnt = hist[bin];
          if (run + cnt >= need) { sh_digit = (uint32_t)bin; sh_need = need - run; break; }
          run += cnt;
        }
      }
    }
    __syncthreads();
    prefix |= sh_digit << shift;
    mask |= 255u << shift;
    need = sh_need;
  }
  const uint32_t tau = prefix;  // key of the M-th largest score; `need` equal keys are kept, lowest index first (R23)
  uint32_t gt_before = 0u, eq_before = 0u;
  for (int base = 0; base < Kpad; base += kSelThreads) {
    const int t = base + tid;
    const uint32_t u = t < K ? key(t) : 0u;
    const bool gt = t < K && u > tau, eq = t < K && u == tau;
    const uint32_t bg = __ballot_sync(0xffffffffu, gt), be = __ballot_sync(0xffffffffu, eq);
    if (lane == 0) warp_tot[warp] = (uint32_t)__popc(bg) | ((uint32_t)__popc(be) << 16);
    __syncthreads();
    if (warp == 0) {
      const uint32_t c = warp_tot[lane];
      uint32_t incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      warp_off[lane] = incl - c;
      if (lane == 31) sh_chunk_tot = incl;
    }
    __syncthreads();
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t off = warp_off[warp];
    const uint32_t g0 = gt_before + (off & 0xffffu) + (uint32_t)__popc(bg & lt);
    const uint32_t e0 = eq_before + (off >> 16) + (uint32_t)__popc(be & lt);
    if (gt) out[g0 + min(e0, need)] = t;
    else if (eq && e0 < need) out[g0 + e0] = t;
    const uint32_t tot = sh_chunk_tot;
    gt_before += tot & 0xffffu;
    eq_before += tot >> 16;
    __syncthreads();
  }
}

cudaError_t launch_select(const omnimem_ctx* ctx, const StepParams& p, const float* psi_v, const float* psi_a,
                          const int32_t* M_v, const int32_t* M_a, int32_t* idx_v, int32_t* idx_a, cudaStream_t st,
                          int* launches) {
  const int segs = p.L * p.Hkv * 2;
  const size_t smem = (size_t)(p.seg_cap_v > p.seg_cap_a ? p.seg_cap_v : p.seg_cap_a) * sizeof(uint32_t);
  ++*launches;
  if (smem <= 225 * 1024) {   // up to 57600 keys (the paper's 48k budget + a 4096-row chunk) stay in shared memory
    cudaError_t e = cudaFuncSetAttribute(select_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    select_kernel<true><<<segs, kSelThreads, smem, st>>>(p, psi_v, psi_a, M_v, M_a, idx_v, idx_a);
  } else {
    select_kernel<false><<<segs, kSelThreads, 0, st>>>(p, psi_v, psi_a, M_v, M_a, idx_v, idx_a);
  }
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------
// Compaction (P:66 prune): dst[l,h,j] = src row of the j-th kept index, K and V, 128-bit copies,
// kTPR threads per row, kR rows in flight per thread.  Also publishes the new row counts.
// ------------------------------------------------------------------------------------------------------------
template <int kTPR, int kR>
__global__ void __launch_bounds__(256) compact_kernel(StepParams p, const uint4* __restrict__ srcK,
                                                      const uint4* __restrict__ srcV, const uint4* __restrict__ chunkK,
                                                      const uint4* __restrict__ chunkV, const int32_t* __restrict__ idx_v,
                                                      const int32_t* __restrict__ idx_a, const int32_t* __restrict__ M_v,
                                                      const int32_t* __restrict__ M_a, uint4* __restrict__ dstK,
                                                      uint4* __restrict__ dstV, int32_t* __restrict__ dst_n_v,
                                                      int32_t* __restrict__ dst_n) {
  constexpr int kRowsPerPass = 256 / kTPR;
  const int l = blockIdx.z, h = blockIdx.y;
  int Mv, Ma;
  clamp_budgets(p, p.n_v[l], p.n[l], M_v[l], M_a[l], Mv, Ma);
  const int total = Mv + Ma;
  if (blockIdx.x == 0 && h == 0 && threadIdx.x == 0) { dst_n_v[l] = Mv; dst_n[l] = total; }
  const int j0 = blockIdx.x * (kRowsPerPass * kR) + threadIdx.x / kTPR;
  if (j0 - (int)(threadIdx.x / kTPR) >= total) return;
  const int sub = threadIdx.x % kTPR;
  const int n_v = p.n_v[l], n = p.n[l];
  const long long lh = (long long)l * p.Hkv + h;
  uint4 vk[kR], vv[kR];
#pragma unroll
  for (int r = 0; r < kR; ++r) {
    const int j = j0 + r * kRowsPerPass;
    if (j < total) {
      const int m = j < Mv ? 0 : 1;
      const int t = m == 0 ? idx_v[lh * p.cache_cap + j] : idx_a[lh * p.cache_cap + (j - Mv)];
      bool in_chunk;
      const int row = seg_row(p, n_v, n, m, t, in_chunk);
      const long long off = in_chunk ? (lh * p.Nn + row) * kTPR + sub : (lh * p.cache_cap + row) * kTPR + sub;
      vk[r] = __ldg((in_chunk ? chunkK : srcK) + off);
      vv[r] = __ldg((in_chunk ? chunkV : srcV) + off);
    }
  }
#pragma unroll
  for (int r = 0; r < kR; ++r) {
    const int j = j0 + r * kRowsPerPass;
    if (j < total) {
      const long long off = (lh * p.cache_cap + j) * kTPR + sub;
      dstK[off] = vk[r];
      dstV[off] = vv[r];
    }
  }
}

cudaError_t launch_compact(const omnimem_ctx* ctx, const StepParams& p, const void* srcK, const void* srcV,
                           const void* chunkK, const void* chunkV, const int32_t* idx_v, const int32_t* idx_a,
                           const int32_t* M_v, const int32_t* M_a, void* dstK, void* dstV, int32_t* dst_n_v,
                           int32_t* dst_n, cudaStream_t st, int* launches) {
  const int row_bytes = p.D * (ctx->cfg.dtype == OMNIMEM_FP32 ? 4 : 2);
  const int tpr = row_bytes / 16;
  constexpr int kR = 4;
  const int rows_per_block = 256 / tpr * kR;
  dim3 grid((p.cache_cap + rows_per_block - 1) / rows_per_block, p.Hkv, p.L);
  ++*launches;
#define OMNIMEM_CP(TPR)                                                                                              \
  compact_kernel<TPR, kR><<<grid, 256, 0, st>>>(p, (const uint4*)srcK, (const uint4*)srcV, (const uint4*)chunkK,    \
                                                (const uint4*)chunkV, idx_v, idx_a, M_v, M_a, (uint4*)dstK,        \
                                                (uint4*)dstV, dst_n_v, dst_n)
  if (tpr == 8) OMNIMEM_CP(8); else if (tpr == 16) OMNIMEM_CP(16); else OMNIMEM_CP(32);
#undef OMNIMEM_CP
  return cudaGetLastError();
}

// Time-interleaved chunk (R25'): from the per-row modality map (0 visual, 1 audio, rows in true temporal order) build
// row_of_seg (rows of the visual tokens in order, then the audio tokens') and seg_of_row ((m << 30) | rank within m).
// One block; thread i owns a contiguous slice, slice counts are scanned in shared memory.
__global__ void __launch_bounds__(1024) chunk_maps_kernel(const int32_t* __restrict__ modality, int Nn, int Nn_v,
                                                          int32_t* __restrict__ row_of_seg,
                                                          int32_t* __restrict__ seg_of_row) {
  __shared__ int cnt[1024];
  const int per = (Nn + 1023) / 1024;
  const int r0 = threadIdx.x * per, r1 = min(Nn, r0 + per);
  int c = 0;
  for (int r = r0; r < r1; ++r) c += modality[r] == 0;
  cnt[threadIdx.x] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    int run = 0;
    for (int i = 0; i < 1024; ++i) { const int v = cnt[i]; cnt[i] = run; run += v; }
  }
  __syncthreads();
  int jv = cnt[threadIdx.x], ja = r0 < Nn ? r0 - jv : 0;   // visual / audio tokens before this slice
  for (int r = r0; r < r1; ++r) {
    const int m = modality[r] == 0 ? 0 : 1;
    const int j = m == 0 ? jv++ : ja++;
    seg_of_row[r] = (m << 30) | j;
    const int slot = m == 0 ? j : Nn_v + j;
    if (slot < Nn && (m == 1 || j < Nn_v)) row_of_seg[slot] = r;   // a map that disagrees with Nn_v cannot write out of bounds
  }
}

cudaError_t launch_chunk_maps(const int32_t* modality, int Nn, int Nn_v, int32_t* row_of_seg, int32_t* seg_of_row,
                              cudaStream_t st, int* launches) {
  if (Nn == 0) return cudaSuccess;
  chunk_maps_kernel<<<1, 1024, 0, st>>>(modality, Nn, Nn_v, row_of_seg, seg_of_row);
  ++*launches;
  return cudaGetLastError();
}

// The retained hidden states follow the kept tokens: dstH[l, j] = row of the j-th kept index of the layer
// (select_scope == 1: every head keeps the same rows, head 0's index list is read).  One warp per row, 512-byte steps.
__global__ void __launch_bounds__(256) compact_hidden_kernel(StepParams p, const uint4* __restrict__ srcH,
                                                             const uint4* __restrict__ chunkH,
                                                             const int32_t* __restrict__ idx_v,
                                                             const int32_t* __restrict__ idx_a,
                                                             const int32_t* __restrict__ M_v,
                                                             const int32_t* __restrict__ M_a, uint4* __restrict__ dstH,
                                                             int row_vecs) {
  const int l = blockIdx.y, lane = threadIdx.x & 31;
  const int j = blockIdx.x * 8 + (threadIdx.x >> 5);
  int Mv, Ma;
  clamp_budgets(p, p.n_v[l], p.n[l], M_v[l], M_a[l], Mv, Ma);
  const int total = Mv + Ma;
  if (j >= total) return;
  const int m = j < Mv ? 0 : 1;
  const long long lh0 = (long long)l * p.Hkv;  // head 0 of the layer
  const int t = m == 0 ? idx_v[lh0 * p.cache_cap + j] : idx_a[lh0 * p.cache_cap + (j - Mv)];
  bool in_chunk;
  const int row = seg_row(p, p.n_v[l], p.n[l], m, t, in_chunk);
  const uint4* src = in_chunk ? chunkH + ((long long)l * p.Nn + row) * row_vecs : srcH + ((long long)l * p.cache_cap + row) * row_vecs;
  uint4* dst = dstH + ((long long)l * p.cache_cap + j) * row_vecs;
  for (int v0 = lane; v0 < row_vecs; v0 += 128) {
    uint4 r[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) if (v0 + 32 * u < row_vecs) r[u] = __ldg(src + v0 + 32 * u);
#pragma unroll
    for (int u = 0; u < 4; ++u) if (v0 + 32 * u < row_vecs) dst[v0 + 32 * u] = r[u];
  }
}

cudaError_t launch_compact_hidden(const omnimem_ctx* ctx, const StepParams& p, const void* srcH, const void* chunkH,
                                  const int32_t* idx_v, const int32_t* idx_a, const int32_t* M_v, const int32_t* M_a,
                                  void* dstH, cudaStream_t st, int* launches) {
  const int row_vecs = p.d_model * (ctx->cfg.dtype == OMNIMEM_FP32 ? 4 : 2) / 16;
  const dim3 grid((unsigned)((p.cache_cap + 7) / 8), (unsigned)p.L);
  ++*launches;
  compact_hidden_kernel<<<grid, 256, 0, st>>>(p, (const uint4*)srcH, (const uint4*)chunkH, idx_v, idx_a, M_v, M_a,
                                              (uint4*)dstH, row_vecs);
  return cudaGetLastError();
}

}  // namespace omnimem
