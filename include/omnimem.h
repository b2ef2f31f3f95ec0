/*
 * omnimem.h -- C ABI of the B200-native OmniMem per-chunk KV-cache compression step.
 *
 * What it computes (arxiv/paper_2606_07577; "P:<n>" = line of PAPER.md, "R<k>" = reading listed in DESIGN.md):
 * each time a chunk of visual + audio tokens is appended to every layer's KV cache (Eq.3) the cache is
 * pruned back to a fixed budget (Eq.4-5) by
 *   1. importance   a_k  = sum over the chunk's queries of softmax attention on key k      (Eq.6)
 *   2. redundancy   s_k  = mean cosine similarity with the adjacent positions               (Eq.7)
 *   3. AVBA         C_m  = H[abar_m](1 - sbar_m)/log K_m  ->  w_v, w_a  ->  M_v, M_a        (Eq.9-12)
 *                   C^(l), B^(l) = Softmax(C/T)[l] (optional per-layer totals)              (Eq.13-14)
 *   4. select       top-M_m of psi_k = a_k^lambda (1 - s_k) per (layer, KV head, modality)  (Eq.8)
 *   5. compact      gather of the kept K/V rows into the fixed-budget cache
 *
 * Conventions
 *   - All pointers are DEVICE pointers unless a comment says HOST.  The caller owns every buffer; the library
 *     allocates no device memory after omnimem_create, frees nothing of the caller's and never synchronises the host
 *     (except omnimem_compress_chunk_host, see there).
 *   - Every call enqueues work on `stream` (a cudaStream_t passed as void*) and returns at once.
 *   - Return value: OMNIMEM_OK or a negative omnimem_status.  Argument errors are detected before any launch.
 *     No C++ exception crosses this boundary.  There is no CPU fallback: on a device that is not sm_100
 *     omnimem_create returns OMNIMEM_UNSUPPORTED.
 *   - Layout of a cache (one per model, "two separate KV caches" of P:56-58 Eq.2 pooled in one buffer):
 *     k, v are [L, Hkv, cache_cap, D] contiguous; for layer l rows [0, n_v[l]) are the visual cache, rows
 *     [n_v[l], n[l]) the audio cache, the same for every KV head of the layer.
 *   - Layout of a chunk: k, v are [L, Hkv, Nn, D], q is [L, Hq, Nn, D], Nn = Nn_v + Nn_a, visual rows first (R25).
 *     Query head j reads KV head j / (Hq/Hkv) (R5).
 *   - Logical key order seen by the attention of Eq.1/Eq.6 (ONE joint softmax, R2):
 *     cached visual, cached audio, new visual, new audio.  Causal inside the chunk (R3): chunk key t is visible to
 *     chunk query i iff t <= i; cached keys are visible to every query.
 *   - Segment-local index t of modality m (the appended sequence K~_m of Eq.3, length K_m = n_m + Nn_m):
 *     t < n_m -> cache row off_m + t (off_v = 0, off_a = n_v);  else chunk row coff_m + (t - n_m) (coff_v = 0,
 *     coff_a = Nn_v).  Per-modality arrays are [L, Hkv, seg_cap_m] fp32 with seg_cap_m = cache_cap + max_chunk_m
 *     (omnimem_seg_cap); entries at t >= K_m are unspecified.
 *   - Budgets (layer_budget, M_v, M_a) are DEVICE arrays: the AVBA split runs on the device every step (R21) and no
 *     call reads them back, so they cannot be rejected on the host.  They are CLAMPED where they are consumed:
 *     a per-layer total B^(l) to [0, cache_cap] in omnimem_allocate / omnimem_compress_chunk, and M_v to
 *     [0, min(K_v, cache_cap)], M_a to [0, min(K_a, cache_cap - M_v)] in omnimem_select / omnimem_compact.  Nothing is
 *     ever written at or beyond row cache_cap of an idx_m or dst row block.  OMNIMEM_CAPACITY is returned only for
 *     sizes the host can see (Nn_v > max_chunk_v, Nn_a > max_chunk_a).
 */
#ifndef OMNIMEM_H_
#define OMNIMEM_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define OMNIMEM_API __attribute__((visibility("default")))
#else
#define OMNIMEM_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  OMNIMEM_OK = 0,
  OMNIMEM_INVALID_ARG = -1,        /* NULL where a pointer is required, negative size, aliasing dst == src ...  */
  OMNIMEM_UNSUPPORTED = -2,        /* dtype / head_dim / device architecture not supported                        */
  OMNIMEM_WORKSPACE_TOO_SMALL = -3,
  OMNIMEM_CUDA_ERROR = -4,         /* details: omnimem_last_cuda_error                                           */
  OMNIMEM_CAPACITY = -5,           /* chunk larger than max_chunk_v / max_chunk_a (host-visible sizes only)       */
  OMNIMEM_STATIC_SCRATCH_EXCEEDED = -6 /* omnimem_redundancy_static only: the problem needs more pair cosines than the
                                      library's built-in array holds (OMNIMEM_STATIC_SCRATCH_FLOATS)              */
} omnimem_status;

enum { OMNIMEM_FP32 = 0, OMNIMEM_BF16 = 1 };

typedef struct omnimem_ctx omnimem_ctx; /* opaque: config, device properties, TMA descriptors, timing events */

typedef struct {
  int32_t n_layers, n_q_heads, n_kv_heads; /* L, Hq, Hkv; Hq % Hkv == 0                                              */
  int32_t head_dim;                        /* D in {64, 128}                                                         */
  int32_t dtype;                           /* OMNIMEM_FP32 (SIMT fp32 path) or OMNIMEM_BF16 (tcgen05 path when D=128) */
  int32_t cache_cap;                       /* rows per (layer, kv head) of each cache buffer (>= every budget)       */
  int32_t max_chunk_v, max_chunk_a;        /* capacity of a chunk per modality                                       */
  float softmax_scale;                     /* c of z = c <q,k>; 0 => 1/sqrt(head_dim) (R4)                           */
  float lambda;                            /* Eq.8; paper default 0.02; 0 = cosine-only ablation     */
  float ratio_r;                           /* Eq.11-12 prior visual:audio ratio; paper default 5             */
  float temperature;                       /* Eq.14 T; paper default 0.2                                     */
  int32_t budget_min, budget_max;          /* Eq.14 clamp [B_min, B_max]; 0,0 => no clamp                    */
  int32_t causal;                          /* 1 = causal inside the chunk (R3, default), 0 = every key visible       */
  int32_t sim_source;                      /* Eq.7 vectors: 0 = value rows (default), 1 = key rows,
                                              2 = the layer's hidden states H (the paper's first form;
                                              needs d_model > 0 and select_scope == 1, R30)                          */
  int32_t sim_stride_v, sim_stride_a;      /* neighbour distance of Eq.7 per modality; 1 = paper literal (R11)       */
  int32_t score_path;                      /* 0 = auto (tcgen05 for bf16 D=128, SIMT otherwise), 1 = force SIMT      */
  int32_t select_scope;                    /* 0 = one index set per (layer, KV head) (north_star, R5);
                                              1 = one index set per layer, the paper-literal reading of P:68-74 where
                                              I carries no head index (R29): psi = (sum_h a)^lambda (1 - mean_h s)         */
  int32_t d_model;                         /* width of the retained hidden states (cache.h, chunk.h); 0 = none;
                                              d_model * element size must be a multiple of 16 bytes                  */
  int32_t score_ctas;                      /* tcgen05 scoring kernels: number of persistent CTAs that share the work
                                              items of a launch; 0 = one per SM (default).  A smaller number leaves SMs
                                              to concurrent work; results do not depend on it                        */
} omnimem_config;

typedef struct {     /* one pooled KV cache */
  void* k;           /* [L, Hkv, cache_cap, D] dtype                                          */
  void* v;           /* [L, Hkv, cache_cap, D] dtype                                          */
  int32_t* n_v;      /* [L] visual rows valid per layer                                       */
  int32_t* n;        /* [L] total rows valid per layer (visual + audio), n[l] <= cache_cap    */
  void* h;           /* sim_source == 2 only, else NULL: [L, cache_cap, d_model] dtype, the retained hidden states
                        H^(l) of the cached tokens, row r belongs to the token of K/V row r (one set of rows per
                        layer: the kept set is the same for every head, select_scope == 1)          */
} omnimem_cache;

typedef struct {     /* one chunk, modality-blocked */
  const void* k;     /* [L, Hkv, Nn, D]                                                       */
  const void* v;     /* [L, Hkv, Nn, D]                                                       */
  const void* q;     /* [L, Hq, Nn, D]  queries = the chunk's tokens                          */
  const float* lse;  /* optional [L, Hq, Nn]: natural-log LSE of the scaled, masked logits of Eq.1 as produced by the
                        model's own attention forward; NULL => computed here (score pass 1)                        */
  int32_t Nn_v, Nn_a; /* HOST ints: rows of each modality in this chunk                       */
  const void* h;     /* sim_source == 2 only, else NULL: [L, Nn, d_model] hidden states of the chunk's tokens */
  const int32_t* modality; /* NULL = modality-blocked chunk (visual rows [0, Nn_v), then audio rows; R25).  Else
                        DEVICE [Nn]: 0 = visual, 1 = audio for every chunk row, rows in TRUE temporal order (a
                        time-interleaved chunk, R25'); exactly Nn_v zeros.  The causal mask of R3 then follows the true
                        position, and the j-th visual (audio) row of the chunk is entry n_v + j (n_a + j) of the
                        appended visual (audio) sequence.  The same map serves every layer.                */
} omnimem_chunk;

typedef struct {     /* outputs of the scoring stages; any pointer may be NULL except where noted */
  float *a_v, *a_a;      /* Eq.6 importance per modality segment  [L, Hkv, seg_cap_m]  (required)  */
  float *s_v, *s_a;      /* Eq.7 redundancy                                             (required)  */
  float *psi_v, *psi_a;  /* Eq.8 score, fp32: the public array that selection consumes  (required)  */
  float* lse_out;        /* [L, Hq, Nn] LSE computed by pass 1 (natural log) or NULL                */
  float* row_entropy;    /* [L, Hq, Nn] -sum_k p ln p per query row (diagnostic, R16) or NULL       */
  double* stats;         /* [L, 8]: Hn_v, Hn_a, sbar_v, sbar_a, C_v, C_a, Hn_all, sbar_all (required) */
} omnimem_scores;

/* ---- life cycle ---------------------------------------------------------------------------------------------- */
/* HOST pointers.  Validates the config, queries the current CUDA device, creates timing events.  *out is set only
 * on success.  Errors: INVALID_ARG (NULL, non-positive sizes, Hq % Hkv != 0, strides < 1), UNSUPPORTED (dtype,
 * head_dim, device is not compute capability 10.x), CUDA_ERROR. */
OMNIMEM_API int omnimem_create(const omnimem_config* cfg, omnimem_ctx** out);
OMNIMEM_API int omnimem_destroy(omnimem_ctx* ctx);
/* Bytes of device scratch every call below needs at this ctx's capacities; the caller allocates it once
 * (256-byte aligned) and passes it to each call.  Contents need not persist between calls. */
OMNIMEM_API size_t omnimem_workspace_bytes(const omnimem_ctx* ctx);
/* Row stride of the per-modality arrays: cache_cap + max_chunk_m (m = 0 visual, 1 audio). */
OMNIMEM_API int32_t omnimem_seg_cap(const omnimem_ctx* ctx, int32_t modality);
OMNIMEM_API const char* omnimem_strerror(int status);              /* static string                                     */
OMNIMEM_API const char* omnimem_last_cuda_error(const omnimem_ctx* ctx); /* cudaGetErrorString of the last CUDA failure  */

/* ---- the step before the path: the chunk's attention forward (Eq.1, Eq.2) ---- */
/* Y_c = MHSA(Q_c, K_c, V_c, O_c, P_c): for every layer l, query head j and chunk query i
 *     y[l, j, i, :] = sum_k softmax_k(c <q_i, k_k>) v_k      over the logical key order of "Conventions"
 * (cached visual, cached audio, chunk rows; ONE joint softmax, R2; causal inside the chunk, R3; query head j reads
 * KV head j / G, R5), and lse_out[l, j, i] = log sum_k exp(c <q_i, k_k>) (natural log) -- exactly the array
 * omnimem_chunk.lse takes, so that omnimem_compress_chunk on the same chunk skips score pass 1: the forward a model
 * runs anyway (Eq.1) makes Eq.6 a single pass over Q K^T.
 * y: DEVICE [L, Hq, Nn, D] of the context dtype (bf16: fp32 accumulation, P rounded to bf16 before P V, Y rounded once:
 * |y - exact| <= 2^-7 sum_k p_k |v_k| element-wise, R32; fp32: 1e-5 of the same magnitude);
 * lse_out: DEVICE float [L, Hq, Nn].  Both required.  chunk->lse, ->h and ->modality are ignored (the mask follows the
 * storage order of the chunk rows, which is the temporal order in both chunk layouts).  bf16 with D = 128 runs on
 * tcgen05 (tensor memory accumulators for S and O, TMA-fed K / V ring); fp32 and D = 64 on a SIMT kernel.
 * Rows n[l] .. cache_cap of the cache buffers are never read into a result.  Nn = 0: nothing is written.
 * The forward uses no workspace: ws may be NULL and ws_bytes 0 (a model that only wants Y and the LSE need not allocate
 * the compression workspace); whatever is passed is ignored.
 * Errors: INVALID_ARG, CAPACITY (Nn_v > max_chunk_v, Nn_a > max_chunk_a), CUDA_ERROR. */
OMNIMEM_API int omnimem_attend(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, void* y, float* lse_out,
                   void* ws, size_t ws_bytes, void* stream);

/* ---- stage 1-3a: importance, redundancy, psi, AVBA statistics (Eq.6-10, Eq.13) ------------------------------- */
/* src, chunk, out: HOST structs holding DEVICE pointers.  Launches: [LSE pass unless chunk->lse] -> column-sum pass
 * -> cosine pass -> finalize (psi, partial statistics) -> statistics.  Errors: INVALID_ARG, CAPACITY (Nn_v > max_chunk_v,
 * Nn_a > max_chunk_a), WORKSPACE_TOO_SMALL, CUDA_ERROR.  An empty chunk (Nn = 0) yields a = 0 and stats from s only. */
OMNIMEM_API int omnimem_score(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, omnimem_scores* out,
                  void* ws, size_t ws_bytes, void* stream);

/* ---- stage 3b: budgets (Eq.11-12; Eq.13-14 when layer_budget == NULL) ---------------------------------------- */
/* stats [L,8] as written by omnimem_score; n_v, n [L]; layer_budget [L] int32 per-layer totals B^(l) (the paper
 * fixes them offline) or NULL => B^(l) = Softmax_l(C^(l)/T) * total_budget, clamped to [budget_min,
 * budget_max], integerised by largest remainder (R19, R20).  Out: M_v, M_a [L] with M_v + M_a = min(B^(l), K_v + K_a),
 * M_m <= K_m (R22); layer_budget_out [L] or NULL receives the totals used (after the clamp to [0, cache_cap]).
 * The bounded split is b_l = clip(kappa pi_l, B_min, B_max) with kappa set by sum_l b_l = total_budget; if
 * total_budget >= L B_max (<= L B_min) every layer gets B_max (B_min). */
OMNIMEM_API int omnimem_allocate(omnimem_ctx* ctx, const double* stats, const int32_t* n_v, const int32_t* n, int32_t Nn_v,
                     int32_t Nn_a, const int32_t* layer_budget, int64_t total_budget, int32_t* M_v, int32_t* M_a,
                     int32_t* layer_budget_out, void* stream);

/* ---- offline calibration of the per-layer totals (Eq.13-14; NEXT-2 of SURVEY.md section 8(f)) ---------- */
/* "The budget is determined offline for each model based on a small calibration set of videos".  Reading R28:
 * the statistics of every calibration chunk (stats [L,8] as written by omnimem_score) are summed into
 * acc [(L+1)*8] doubles (DEVICE, zeroed by the caller before the first chunk; acc[8 l + i] = sum of statistic i of layer
 * l, acc[8 L] = number of chunks); omnimem_calibrate_budgets writes their arithmetic means to mean_stats_out [L,8]
 * (DEVICE) and B^(l) = Softmax_l(C^(l)/T) * total_budget with C^(l) = mean Hn_all * (1 - mean sbar_all) (Eq.13-14,
 * clamp and rounding as in omnimem_allocate, R19-R20) to layer_budget_out [L] (DEVICE), the table that
 * omnimem_compress_chunk takes as `layer_budget`.  Errors: INVALID_ARG, CUDA_ERROR. */
OMNIMEM_API int omnimem_calibrate_accumulate(omnimem_ctx* ctx, const double* stats, double* acc, void* stream);
OMNIMEM_API int omnimem_calibrate_budgets(omnimem_ctx* ctx, const double* acc, int64_t total_budget, double* mean_stats_out,
                              int32_t* layer_budget_out, void* stream);

/* ---- stage 4: segmented top-M (Eq.4-5) ---------------------------------------------------------------- */
/* psi_m [L, Hkv, seg_cap_m] fp32 (finite); per (l, h, m) writes the segment-local indices of the M_m[l] largest
 * psi to idx_m[l, h, 0:M_m[l]) in ASCENDING index order; among equal psi the lowest index wins (R23).
 * idx_m are [L, Hkv, cache_cap] int32; entries at >= M_m[l] are left untouched.  M_m are clamped as stated under
 * "Budgets" above. */
OMNIMEM_API int omnimem_select(omnimem_ctx* ctx, const float* psi_v, const float* psi_a, const int32_t* n_v, const int32_t* n,
                   int32_t Nn_v, int32_t Nn_a, const int32_t* M_v, const int32_t* M_a, int32_t* idx_v, int32_t* idx_a,
                   void* ws, size_t ws_bytes, void* stream);

/* ---- stage 5: prune / gather-compaction ---------------------------------------------------------- */
/* dst[l,h,0:M_v] = visual rows idx_v, dst[l,h,M_v:M_v+M_a] = audio rows idx_a, K and V, byte-exact;
 * dst->n_v[l] = M_v[l], dst->n[l] = M_v[l] + M_a[l].  dst buffers must not alias src's (INVALID_ARG if
 * dst->k == src->k or dst->v == src->v): the caller ping-pongs two caches.  With sim_source == 2 the retained hidden
 * states follow the kept tokens too: dst->h[l, j] = the hidden row of the j-th kept token of layer l (head 0's index
 * list; select_scope == 1 makes every head's list the same).  chunk->modality, when set, is honoured (R25').
 * The context's small device scratch for the interleaving maps is reused by every call: one stream per context. */
OMNIMEM_API int omnimem_compact(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, const int32_t* idx_v,
                    const int32_t* idx_a, const int32_t* M_v, const int32_t* M_a, omnimem_cache* dst, void* stream);

/* ---- the fused step: stages 1-5 for all layers, one stream, no host synchronisation ------------------------------- */
/* layer_budget [L] device int32 (required).  opt_out NULL => scores live in ws; opt_idx_* NULL => indices live in ws.
 * opt_M_v / opt_M_a [L] or NULL.  When opt_out is NULL, layers with nothing to evict (n[l] + Nn <= layer_budget[l])
 * skip the scoring passes: their rows are appended unchanged. */
OMNIMEM_API int omnimem_compress_chunk(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk,
                           const int32_t* layer_budget, omnimem_cache* dst, omnimem_scores* opt_out,
                           int32_t* opt_idx_v, int32_t* opt_idx_a, int32_t* opt_M_v, int32_t* opt_M_a, void* ws,
                           size_t ws_bytes, void* stream);

/* ---- the fused step fed from HOST memory (end-to-end entry) --------------------------------------------------- */
/* host_chunk->k/v/q (and ->lse if non-NULL) are HOST pointers (pinned memory for full copy speed) with the chunk
 * layout above; dev_chunk holds DEVICE staging buffers of the same shapes (caller-owned).  Copies the chunk to the
 * device, runs the fused step, copies M_v, M_a back to the HOST arrays host_M_v, host_M_a [L] (pinned) and
 * synchronises `stream` before returning.  Layers are independent through the whole step (the per-layer
 * totals are an input, R21), so the chunk is copied and compressed in up to 8 groups of consecutive layers (1, 2, 3, 4, 6, 9, ... layers): the
 * copies run on a stream owned by the context (ordered after everything already enqueued on `stream`) and the
 * kernels of group g on `stream` overlap the copy of group g + 1.  host_chunk->h and host_chunk->modality, when set,
 * are HOST arrays too and dev_chunk->h / dev_chunk->modality their DEVICE staging buffers.  Results are identical to omnimem_compress_chunk
 * on the same inputs.  Returns the byte counts moved through h2d_bytes / d2h_bytes (HOST, may be NULL).  All argument
 * errors are detected before anything is enqueued; if a CUDA call fails later, both streams are synchronised before the
 * status is returned, so the host buffers are no longer being read.  Per-stage timing (omnimem_get_stage_ms) after this
 * entry covers the LAST layer group only (the events are re-recorded per group). */
OMNIMEM_API int omnimem_compress_chunk_host(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* host_chunk,
                                const omnimem_chunk* dev_chunk, const int32_t* layer_budget, omnimem_cache* dst,
                                int32_t* host_M_v, int32_t* host_M_a, int64_t* h2d_bytes, int64_t* d2h_bytes,
                                void* ws, size_t ws_bytes, void* stream);

/* ---- Eq.7 redundancy without any allocation ------------------------------------------------------ */
/* Who this is for.  Everything above assumes the caller can obtain device memory: omnimem_create itself calls cudaMalloc
 * (work counters, interleaving maps) and every stage wants a workspace of omnimem_workspace_bytes.  Some users of this
 * library cannot do that at the point where they need the scores.  Two we know of: (1) a serving engine that handed all
 * of HBM to its own paged KV-cache pool at start-up, so a later cudaMalloc either fails outright or, when it succeeds,
 * stalls every stream of the device while the driver maps memory in the middle of serving; (2) an operator body that runs
 * inside a host runtime's callback, is given its input and output tensors and nothing else, and is forbidden to allocate
 * there.  For them this ONE call computes the redundancy term of the score with no context, no workspace and no
 * cudaMalloc / cudaFree / allocating library routine on any path: the intermediate pair cosines live in an array that is
 * part of the library image.
 *
 * What it computes: s_m[l, h, t] = mean over the neighbours t +- sim_stride_m that exist inside the appended sequence of
 * modality m (Eq.3) of cos(x_t, x_neighbour), clamped to [-1, 1], 0 when there is no neighbour -- the same numbers
 * omnimem_score writes to omnimem_scores.s_v / .s_a.  x are the rows of cache_x [L, Hkv, cache_cap, D] and chunk_x
 * [L, Hkv, Nn, D] (pass the value buffers for the paper's default, or the key buffers), dtype OMNIMEM_FP32 or
 * OMNIMEM_BF16, D in {64, 128}, segment conventions as at the top of this header, chunk modality-blocked (visual rows
 * first).  n_v, n: DEVICE int32 [L].  Nn_v, Nn_a: HOST ints, Nn_m <= max_chunk_m.  s_v, s_a: DEVICE float
 * [L, Hkv, cache_cap + max_chunk_m], caller-owned like every input; entries at t >= K_m are left untouched.
 * All work is enqueued on `stream`, which must belong to the CURRENT device; the call does not wait for it.
 *
 * The limit.  The built-in array holds OMNIMEM_STATIC_SCRATCH_FLOATS = 2^20 floats (4 MiB; every GPU that loads the
 * library carries it until the process exits).  One float is needed per (layer, KV head, row at full capacity):
 *     n_layers * n_kv_heads * (2 * cache_cap + max_chunk_v + max_chunk_a)  <=  OMNIMEM_STATIC_SCRATCH_FLOATS,
 * else OMNIMEM_STATIC_SCRATCH_EXCEEDED is returned before anything is launched.  Layers are independent, so a larger
 * model is served by one call per group of layers (config 2's shape: 6 layers per call) with the pointers advanced.
 *
 * Sharing.  There is one array per device and every call on that device uses it.  Calls issued to the same stream run one
 * after the other and are safe.  Two calls that can be on the GPU at the same time (different streams, different host
 * threads) overwrite each other's intermediates: serialise them yourself (one stream, or an event between them).  The
 * array keeps the previous call's contents; nothing has to be cleared, because every entry a call reads it has written
 * first.
 *
 * First call.  The first call on each device looks up where the array lives on that device (cudaGetSymbolAddress, once,
 * under a lock, with that device current) and may make the CUDA runtime load this library's device code.  Make that first
 * call during start-up, before any stream capture begins; later calls only launch two kernels.
 * Errors: INVALID_ARG (NULL pointer, non-positive size, stride < 1), UNSUPPORTED (dtype, head_dim, device is not compute
 * capability 10.x), CAPACITY (Nn_m > max_chunk_m), STATIC_SCRATCH_EXCEEDED, CUDA_ERROR (a runtime call or launch failed). */
#define OMNIMEM_STATIC_SCRATCH_FLOATS (1 << 20)
OMNIMEM_API int omnimem_redundancy_static(int32_t dtype, int32_t n_layers, int32_t n_kv_heads, int32_t head_dim,
                              int32_t cache_cap, int32_t max_chunk_v, int32_t max_chunk_a, int32_t sim_stride_v,
                              int32_t sim_stride_a, const void* cache_x, const int32_t* n_v, const int32_t* n,
                              const void* chunk_x, int32_t Nn_v, int32_t Nn_a, float* s_v, float* s_a, void* stream);

/* ---- per-stage device timing (CUDA events on `stream`, recorded inside the calls above when enabled) ---------- */
enum {
  OMNIMEM_STAGE_LSE = 0,      /* score pass 1 */
  OMNIMEM_STAGE_COLSUM = 1,   /* score pass 2 */
  OMNIMEM_STAGE_COSINE = 2,
  OMNIMEM_STAGE_FINALIZE = 3, /* psi + statistics */
  OMNIMEM_STAGE_ALLOCATE = 4,
  OMNIMEM_STAGE_SELECT = 5,
  OMNIMEM_STAGE_COMPACT = 6,
  OMNIMEM_STAGE_ATTEND = 7,   /* omnimem_attend (not part of the fused step) */
  OMNIMEM_N_STAGES = 8
};
OMNIMEM_API int omnimem_set_profiling(omnimem_ctx* ctx, int32_t enabled);
/* HOST out[OMNIMEM_N_STAGES]: milliseconds of each stage in the most recent call (0 for stages that did not run);
 * synchronises on the recorded events.  launches_out (HOST, may be NULL): kernels launched by that call. */
OMNIMEM_API int omnimem_get_stage_ms(omnimem_ctx* ctx, float* out, int32_t* launches_out);

#ifdef __cplusplus
}
#endif
#endif /* OMNIMEM_H_ */
