// Shared declarations of the CUDA path (host context, kernel parameter block, segment maps).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/omnimem.h"

namespace omnimem {

// Kernel parameter block (by value).  Names follow include/omnimem.h and the paper's notation.
struct StepParams {
  int L, Hq, Hkv, G, D;
  int cache_cap;
  int Nn_v, Nn_a, Nn;        // this chunk
  int seg_cap_v, seg_cap_a;  // row strides of the per-modality arrays
  int causal;
  int stride_v, stride_a;    // Eq.7 neighbour distance per modality
  float scale;               // c
  float scale_log2e;         // c * log2(e)
  float lambda;
  int shared_heads;  // select_scope == 1: one score per token and layer (R29)
  int d_model;       // width of the hidden-state rows (sim_source == 2), else 0
  // device state
  const int32_t* n_v;        // [L]
  const int32_t* n;          // [L]
  const int32_t* skip_budget;  // [L] or nullptr: layers with n[l] + Nn <= skip_budget[l] skip scoring
  // time-interleaved chunk (chunk.modality != NULL, R25'), else nullptr = modality-blocked chunk:
  const int32_t* row_of_seg;   // [Nn]: chunk rows of the visual tokens in order, then those of the audio tokens
  const int32_t* seg_of_row;   // [Nn]: (modality << 30) | index among the chunk's tokens of that modality
};

// Segment maps (include/omnimem.h "Conventions"; Eq.3 appended sequences).
__host__ __device__ __forceinline__ int seg_len(const StepParams& p, int n_v, int n, int m) {
  return m == 0 ? n_v + p.Nn_v : (n - n_v) + p.Nn_a;
}
// segment-local t -> row in cache (in_chunk = false) or chunk (in_chunk = true)
__device__ __forceinline__ int seg_row(const StepParams& p, int n_v, int n, int m, int t, bool& in_chunk) {
  const int n_m = m == 0 ? n_v : n - n_v;
  if (t < n_m) {
    in_chunk = false;
    return (m == 0 ? 0 : n_v) + t;
  }
  in_chunk = true;
  const int j = (m == 0 ? 0 : p.Nn_v) + (t - n_m);
  return p.row_of_seg ? p.row_of_seg[j] : j;
}
// logical key (cache row r < n, or chunk row) -> (modality, segment-local index)
__device__ __forceinline__ void cache_row_to_seg(int n_v, int r, int& m, int& t) {
  if (r < n_v) { m = 0; t = r; } else { m = 1; t = r - n_v; }
}
__device__ __forceinline__ void chunk_row_to_seg(const StepParams& p, int n_v, int n, int r, int& m, int& t) {
  if (p.seg_of_row) {
    const int e = p.seg_of_row[r];
    m = e >> 30;
    t = (m == 0 ? n_v : n - n_v) + (e & 0x3FFFFFFF);
    return;
  }
  if (r < p.Nn_v) { m = 0; t = n_v + r; } else { m = 1; t = (n - n_v) + (r - p.Nn_v); }
}
// Budgets are device data (AVBA runs on the device, R21; the public stage calls take device arrays): nothing on the
// host can validate them, so select / compact clamp them to the rows that exist and to what one cache row block holds.
// With in-range budgets (what allocate produces) this is the identity.
__device__ __forceinline__ void clamp_budgets(const StepParams& p, int n_v, int n, int mv_in, int ma_in, int& Mv, int& Ma) {
  const int Kv = seg_len(p, n_v, n, 0), Ka = seg_len(p, n_v, n, 1);
  Mv = min(max(mv_in, 0), min(Kv, p.cache_cap));
  Ma = min(max(ma_in, 0), min(Ka, p.cache_cap - Mv));
}
__device__ __forceinline__ bool layer_skips_scoring(const StepParams& p, int l) {
  return p.skip_budget != nullptr && p.n[l] + p.Nn <= p.skip_budget[l];
}

// Buffers of one step (device pointers).
struct StepBuffers {
  const void *cacheK, *cacheV, *chunkK, *chunkV, *Q;
  const void *cacheH, *chunkH;  // hidden states (sim_source == 2) or nullptr
  const float* lse_in;   // caller-supplied natural-log LSE [L,Hq,Nn] or nullptr
  float* lse;            // SIMT path: natural-log LSE read by pass 2 (== lse_in when supplied)
  float* lse2;           // tcgen05 path: internal log2-domain LSE, rows padded to a multiple of 128
  float* lse_out;        // caller's natural-log output or nullptr
  float* row_entropy;    // or nullptr
  float *a_v, *a_a, *s_v, *s_a, *psi_v, *psi_a;
  float *la_v, *la_a;    // internal: log2 of the importance of the keys whose fp32 sum is below 2^-100 (R31), [L,Hkv,seg_cap_m]
  int32_t* rescue_items; // tcgen05 path: [1 + items of pass 2] count + list of the items redone in the log domain (R31)
  float* cosn;           // [L,Hkv,seg_cap_v+seg_cap_a]: cos(x_t, x_{t+sigma})
  double* partials;      // [L][2][nblk][3]
  double* stats;         // [L,8]
};

struct TmaMaps;  // score_tc.cu

}  // namespace omnimem

#define OMNIMEM_HOST_GROUPS 8   // layer groups of the pipelined host entry

struct omnimem_ctx {
  omnimem_config cfg;
  int device;
  int sm_count;
  int cc_major, cc_minor;
  int seg_cap_v, seg_cap_a;
  int fin_blocks;  // blocks per (layer, modality) of the finalize kernel
  float scale;
  bool use_tc;
  cudaError_t last_err;
  bool profiling;
  cudaEvent_t ev[2 * OMNIMEM_N_STAGES];
  bool ev_used[OMNIMEM_N_STAGES];
  int launches;
  void* encode_tiled;  // cuTensorMapEncodeTiled entry point
  int32_t* sched;        // device [4]: work-item counters of the persistent scoring kernels (zeroed before each launch)
  int32_t* chunk_maps;   // device [2 * (max_chunk_v + max_chunk_a)]: row_of_seg, seg_of_row of an interleaved chunk
  cudaStream_t copy_stream;                        // omnimem_compress_chunk_host: host -> device copies of the next layer group
  cudaEvent_t ev_copy[OMNIMEM_HOST_GROUPS + 1];    // [g] group g is on the device; [last] `stream` reached the call
};

namespace omnimem {

// launchers (each returns cudaGetLastError() after its launches; `launches` is incremented per kernel)
cudaError_t launch_lse_simt(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_colsum_simt(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_lse_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_colsum_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_attend_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, void* y, float* lse_nat,
                             cudaStream_t st, int* launches);
cudaError_t launch_attend_simt(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, void* y, float* lse_nat,
                               cudaStream_t st, int* launches);
cudaError_t launch_colsum_rescue(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_colsum_rescue_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_cosine(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_finalize(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches);
cudaError_t launch_allocate(const omnimem_ctx* ctx, const StepParams& p, const double* stats, const int32_t* layer_budget,
                            int64_t total_budget, int32_t* M_v, int32_t* M_a, int32_t* layer_budget_out, cudaStream_t st,
                            int* launches);
cudaError_t launch_chunk_maps(const int32_t* modality, int Nn, int Nn_v, int32_t* row_of_seg, int32_t* seg_of_row,
                              cudaStream_t st, int* launches);
cudaError_t launch_compact_hidden(const omnimem_ctx* ctx, const StepParams& p, const void* srcH, const void* chunkH,
                                  const int32_t* idx_v, const int32_t* idx_a, const int32_t* M_v, const int32_t* M_a,
                                  void* dstH, cudaStream_t st, int* launches);
cudaError_t launch_calib_accumulate(int L, const double* stats, double* acc, cudaStream_t st, int* launches);
cudaError_t launch_calib_mean(int L, const double* acc, double* mean, cudaStream_t st, int* launches);
cudaError_t launch_select(const omnimem_ctx* ctx, const StepParams& p, const float* psi_v, const float* psi_a,
                          const int32_t* M_v, const int32_t* M_a, int32_t* idx_v, int32_t* idx_a, cudaStream_t st,
                          int* launches);
cudaError_t launch_compact(const omnimem_ctx* ctx, const StepParams& p, const void* srcK, const void* srcV,
                           const void* chunkK, const void* chunkV, const int32_t* idx_v, const int32_t* idx_a,
                           const int32_t* M_v, const int32_t* M_a, void* dstK, void* dstV, int32_t* dst_n_v,
                           int32_t* dst_n, cudaStream_t st, int* launches);

}  // namespace omnimem
