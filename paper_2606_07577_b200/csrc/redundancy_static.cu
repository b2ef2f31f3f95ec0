// omnimem_redundancy_static: Eq.7 redundancy (value rows per P:103) for callers that cannot allocate device memory.
//
// The regular route to s_v / s_a is omnimem_score: cosine_kernel writes cos(x_t, x_{t+sigma}) for every row into a scratch
// array ("cosn") carved from the caller's workspace and finalize_kernel turns it into the neighbour mean.  That route
// needs a context (omnimem_create calls cudaMalloc) and a workspace the caller got from cudaMalloc.  Here the same two
// steps run with the pair cosines in a fixed array that is part of the library image, so nothing is allocated by anyone:
// no context, no workspace, no cudaMalloc / cudaFree / allocating library call anywhere below.
//
// The array is one per device and shared by every call (see the header for what that means for concurrent callers).
#include <mutex>

#include "common.cuh"

// The scratch itself: OMNIMEM_STATIC_SCRATCH_FLOATS fp32 pair cosines = 4 MiB, resident on every GPU that loads the
// library until the process exits.  In HOST code this name is only a handle for the runtime (it is not a device address and
// must never be handed to a kernel); scratch_address() below asks the runtime for the real per-device address.
static __device__ __align__(256) float g_pair_cos[OMNIMEM_STATIC_SCRATCH_FLOATS];

namespace {

using omnimem::StepParams;

constexpr int kMaxDevices = 64;
struct DeviceSetup {
  float* pair_cos = nullptr;   // device address of g_pair_cos on this device
  int cc_major = 0;
};
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

// Once per device, with that device current: resolve where g_pair_cos lives on it.
cudaError_t scratch_address(int dev, DeviceSetup* out) {
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  DeviceSetup& s = g_setup[dev];
  if (s.pair_cos == nullptr) {
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return e;
    float* ptr = nullptr;
    if (major == 10) {   // the image holds sm_100a code only: on anything else there is no copy of the array to find
      e = cudaGetSymbolAddress((void**)&ptr, g_pair_cos);
      if (e != cudaSuccess) return e;
      if (ptr == nullptr) return cudaErrorInvalidSymbol;
    }
    s.cc_major = major;
    s.pair_cos = ptr;
  }
  *out = s;
  return cudaSuccess;
}

__device__ __forceinline__ void acc16(const uint4& x, const uint4& y, float& dot, float& nx, float& ny, float) {
  const float xs[4] = {__uint_as_float(x.x), __uint_as_float(x.y), __uint_as_float(x.z), __uint_as_float(x.w)};
  const float ys[4] = {__uint_as_float(y.x), __uint_as_float(y.y), __uint_as_float(y.z), __uint_as_float(y.w)};
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    dot = fmaf(xs[e], ys[e], dot);
    nx = fmaf(xs[e], xs[e], nx);
    ny = fmaf(ys[e], ys[e], ny);
  }
}
// bf16: products of two bf16 values are exact in fp32, so widening first loses nothing; even and odd elements keep
// separate running sums (the order the regular cosine_kernel uses)
__device__ __forceinline__ void acc16(const uint4& x, const uint4& y, float& dot, float& nx, float& ny, __nv_bfloat16) {
  const uint32_t xs[4] = {x.x, x.y, x.z, x.w}, ys[4] = {y.x, y.y, y.z, y.w};
  float d1 = 0.f, nx1 = 0.f, ny1 = 0.f;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    const float xl = __uint_as_float(xs[e] << 16), xh = __uint_as_float(xs[e] & 0xffff0000u);
    const float yl = __uint_as_float(ys[e] << 16), yh = __uint_as_float(ys[e] & 0xffff0000u);
    dot = fmaf(xl, yl, dot); d1 = fmaf(xh, yh, d1);
    nx = fmaf(xl, xl, nx);   nx1 = fmaf(xh, xh, nx1);
    ny = fmaf(yl, yl, ny);   ny1 = fmaf(yh, yh, ny1);
  }
  dot += d1; nx += nx1; ny += ny1;
}

// pair_cos[lh, out(m, t)] = cos(x_t, x_{t+sigma_m}) for every row t of modality m that has a partner inside its appended
// sequence (Eq.3).  Four threads share a row, 16 bytes at a time; blockIdx.x = (layer, KV head), blockIdx.y strides over
// the rows that exist.  Every entry the second kernel reads is written here first, so the array never has to be cleared.
template <typename T>
__global__ void __launch_bounds__(256) pair_cosine_static_kernel(StepParams p, const T* __restrict__ cacheX,
                                                                 const T* __restrict__ chunkX,
                                                                 float* __restrict__ pair_cos) {
  constexpr int kTPR = 4, kRows = 256 / kTPR;
  const int items = p.seg_cap_v + p.seg_cap_a;
  const long long lh = blockIdx.x;
  const int l = (int)(lh / p.Hkv);
  const int sub = threadIdx.x % kTPR;
  const int n_v = p.n_v[l], n = p.n[l];
  const int Kv = omnimem::seg_len(p, n_v, n, 0), Ka = omnimem::seg_len(p, n_v, n, 1);
  const int row_vecs = p.D * (int)sizeof(T) / 16;
  const uint4* cbase = reinterpret_cast<const uint4*>(cacheX + lh * p.cache_cap * p.D);
  const uint4* kbase = reinterpret_cast<const uint4*>(chunkX + lh * p.Nn * p.D);
  for (int d0 = blockIdx.y * kRows; d0 < Kv + Ka; d0 += gridDim.y * kRows) {
    const int d = d0 + threadIdx.x / kTPR;   // dense item number: the visual rows, then the audio rows
    const int m = d < Kv ? 0 : 1;
    const int t = m == 0 ? d : d - Kv;
    const int sg = m == 0 ? p.stride_v : p.stride_a;
    const bool active = d < Kv + Ka && t + sg < (m == 0 ? Kv : Ka);
    float dot = 0.f, nx = 0.f, ny = 0.f;
    if (active) {
      bool cx, cy;
      const int rx = omnimem::seg_row(p, n_v, n, m, t, cx), ry = omnimem::seg_row(p, n_v, n, m, t + sg, cy);
      const uint4* x = (cx ? kbase : cbase) + (long long)rx * row_vecs;
      const uint4* y = (cy ? kbase : cbase) + (long long)ry * row_vecs;
      for (int i = sub; i < row_vecs; i += kTPR) acc16(__ldg(x + i), __ldg(y + i), dot, nx, ny, T());
    }
#pragma unroll
    for (int o = kTPR / 2; o; o >>= 1) {
      dot += __shfl_xor_sync(0xffffffffu, dot, o);
      nx += __shfl_xor_sync(0xffffffffu, nx, o);
      ny += __shfl_xor_sync(0xffffffffu, ny, o);
    }
    if (active && sub == 0)
      pair_cos[lh * items + (m == 0 ? t : p.seg_cap_v + t)] = dot / fmaxf(sqrtf(nx) * sqrtf(ny), 1e-8f);  // R12
  }
}

// s_t = mean of the cosines with the neighbours that exist (t + sigma, t - sigma), clamped to [-1, 1]; no neighbour -> 0
// (Eq.7; R10, R12).  blockIdx.x = (layer, KV head), blockIdx.y = modality, blockIdx.z strides over the rows.
__global__ void __launch_bounds__(256) neighbour_mean_static_kernel(StepParams p, const float* __restrict__ pair_cos,
                                                                    float* __restrict__ s_v, float* __restrict__ s_a) {
  const long long lh = blockIdx.x;
  const int l = (int)(lh / p.Hkv), m = blockIdx.y;
  const int n_v = p.n_v[l], n = p.n[l];
  const int Km = omnimem::seg_len(p, n_v, n, m);
  const int cap = m == 0 ? p.seg_cap_v : p.seg_cap_a;
  const int sg = m == 0 ? p.stride_v : p.stride_a;
  const float* cs = pair_cos + lh * (p.seg_cap_v + p.seg_cap_a) + (m == 0 ? 0 : p.seg_cap_v);
  float* s_out = (m == 0 ? s_v : s_a) + lh * cap;
  for (int t = blockIdx.z * 256 + threadIdx.x; t < Km; t += gridDim.z * 256) {
    float sum = 0.f;
    int cnt = 0;
    if (t + sg < Km) { sum += cs[t]; ++cnt; }
    if (t - sg >= 0) { sum += cs[t - sg]; ++cnt; }
    const float s = cnt == 2 ? 0.5f * sum : sum;
    s_out[t] = fminf(1.f, fmaxf(-1.f, s));
  }
}

}  // namespace

extern "C" int omnimem_redundancy_static(int32_t dtype, int32_t n_layers, int32_t n_kv_heads, int32_t head_dim,
                                         int32_t cache_cap, int32_t max_chunk_v, int32_t max_chunk_a,
                                         int32_t sim_stride_v, int32_t sim_stride_a, const void* cache_x,
                                         const int32_t* n_v, const int32_t* n, const void* chunk_x, int32_t Nn_v,
                                         int32_t Nn_a, float* s_v, float* s_a, void* stream) {
  if (n_layers <= 0 || n_kv_heads <= 0 || cache_cap <= 0 || max_chunk_v < 0 || max_chunk_a < 0 || sim_stride_v < 1 ||
      sim_stride_a < 1 || Nn_v < 0 || Nn_a < 0 || !cache_x || !n_v || !n || !s_v || !s_a)
    return OMNIMEM_INVALID_ARG;
  if (Nn_v + Nn_a > 0 && !chunk_x) return OMNIMEM_INVALID_ARG;
  if (dtype != OMNIMEM_FP32 && dtype != OMNIMEM_BF16) return OMNIMEM_UNSUPPORTED;
  if (head_dim != 64 && head_dim != 128) return OMNIMEM_UNSUPPORTED;
  if (Nn_v > max_chunk_v || Nn_a > max_chunk_a) return OMNIMEM_CAPACITY;
  // the limit: one pair cosine per (layer, KV head, row of either appended sequence at full capacity)
  const long long items = 2LL * cache_cap + max_chunk_v + max_chunk_a;
  const long long lh_count = (long long)n_layers * n_kv_heads;
  if (items > INT32_MAX || lh_count * items > (long long)OMNIMEM_STATIC_SCRATCH_FLOATS) return OMNIMEM_STATIC_SCRATCH_EXCEEDED;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return OMNIMEM_CUDA_ERROR;
  if (dev < 0 || dev >= kMaxDevices) return OMNIMEM_UNSUPPORTED;
  DeviceSetup setup;
  e = scratch_address(dev, &setup);
  if (e != cudaSuccess) return OMNIMEM_CUDA_ERROR;
  if (setup.cc_major != 10) return OMNIMEM_UNSUPPORTED;   // sm_100a code only, as everywhere in this library

  StepParams p{};
  p.L = n_layers; p.Hq = n_kv_heads; p.Hkv = n_kv_heads; p.G = 1; p.D = head_dim;
  p.cache_cap = cache_cap;
  p.Nn_v = Nn_v; p.Nn_a = Nn_a; p.Nn = Nn_v + Nn_a;
  p.seg_cap_v = cache_cap + max_chunk_v; p.seg_cap_a = cache_cap + max_chunk_a;
  p.stride_v = sim_stride_v; p.stride_a = sim_stride_a;
  p.n_v = n_v; p.n = n;
  cudaStream_t st = (cudaStream_t)stream;
  const int row_blocks = (int)((items + 63) / 64);
  const dim3 grid1((unsigned)lh_count, (unsigned)(row_blocks < 1024 ? row_blocks : 1024));
  if (dtype == OMNIMEM_FP32)
    pair_cosine_static_kernel<float><<<grid1, 256, 0, st>>>(p, (const float*)cache_x, (const float*)chunk_x, setup.pair_cos);
  else
    pair_cosine_static_kernel<__nv_bfloat16><<<grid1, 256, 0, st>>>(p, (const __nv_bfloat16*)cache_x,
                                                                    (const __nv_bfloat16*)chunk_x, setup.pair_cos);
  e = cudaGetLastError();
  if (e != cudaSuccess) return OMNIMEM_CUDA_ERROR;
  const int seg_cap = p.seg_cap_v > p.seg_cap_a ? p.seg_cap_v : p.seg_cap_a;
  const int blocks2 = (seg_cap + 255) / 256;
  const dim3 grid2((unsigned)lh_count, 2u, (unsigned)(blocks2 < 1024 ? blocks2 : 1024));
  neighbour_mean_static_kernel<<<grid2, 256, 0, st>>>(p, setup.pair_cos, s_v, s_a);
  e = cudaGetLastError();
  return e == cudaSuccess ? OMNIMEM_OK : OMNIMEM_CUDA_ERROR;
}
