// C ABI of the OmniMem compression step (include/omnimem.h): context, validation, workspace carving, launch order.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "common.cuh"

using namespace omnimem;

namespace {

struct WsLayout {
  size_t lse, cosn, partials, a_v, a_a, la_v, la_a, s_v, s_a, psi_v, psi_a, stats, M_v, M_a, idx_v, idx_a, rescue_items, total;
};

size_t align_up(size_t x) { return (x + 255) & ~size_t(255); }

WsLayout ws_layout(const omnimem_ctx* c) {
  const omnimem_config& g = c->cfg;
  const size_t L = g.n_layers, Hq = g.n_q_heads, Hkv = g.n_kv_heads;
  const size_t Nn = (size_t)g.max_chunk_v + g.max_chunk_a;
  WsLayout w{};
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  w.lse = take(L * Hq * ((Nn + 127) / 128 * 128) * sizeof(float));
  w.cosn = take(L * Hkv * ((size_t)c->seg_cap_v + c->seg_cap_a) * sizeof(float));
  w.partials = take(L * 2 * (size_t)c->fin_blocks * 3 * sizeof(double));
  w.a_v = take(L * Hkv * (size_t)c->seg_cap_v * sizeof(float));
  w.a_a = take(L * Hkv * (size_t)c->seg_cap_a * sizeof(float));
  w.la_v = take(L * Hkv * (size_t)c->seg_cap_v * sizeof(float));
  w.la_a = take(L * Hkv * (size_t)c->seg_cap_a * sizeof(float));
  w.s_v = take(L * Hkv * (size_t)c->seg_cap_v * sizeof(float));
  w.s_a = take(L * Hkv * (size_t)c->seg_cap_a * sizeof(float));
  w.psi_v = take(L * Hkv * (size_t)c->seg_cap_v * sizeof(float));
  w.psi_a = take(L * Hkv * (size_t)c->seg_cap_a * sizeof(float));
  w.stats = take(L * 8 * sizeof(double));
  w.M_v = take(L * sizeof(int32_t));
  w.M_a = take(L * sizeof(int32_t));
  w.idx_v = take(L * Hkv * (size_t)g.cache_cap * sizeof(int32_t));
  w.idx_a = take(L * Hkv * (size_t)g.cache_cap * sizeof(int32_t));
  // count + list of pass 2's 256-key items that the log-domain rescue redoes (consumed inside the call that writes it)
  w.rescue_items = take((1 + L * Hkv * (((size_t)g.cache_cap + 255) / 256 + (Nn + 255) / 256)) * sizeof(int32_t));
  w.total = off;
  return w;
}

int fail_cuda(omnimem_ctx* c, cudaError_t e) {
  c->last_err = e;
  return OMNIMEM_CUDA_ERROR;
}

StepParams make_params(const omnimem_ctx* c, int Nn_v, int Nn_a, const int32_t* n_v, const int32_t* n,
                       const int32_t* skip_budget, int n_layers = -1) {
  const omnimem_config& g = c->cfg;
  StepParams p{};
  // a layer range [l0, l0 + L): every per-layer pointer is offset by the caller
  p.L = n_layers < 0 ? g.n_layers : n_layers; p.Hq = g.n_q_heads; p.Hkv = g.n_kv_heads; p.G = g.n_q_heads / g.n_kv_heads; p.D = g.head_dim;
  p.cache_cap = g.cache_cap;
  p.Nn_v = Nn_v; p.Nn_a = Nn_a; p.Nn = Nn_v + Nn_a;
  p.seg_cap_v = c->seg_cap_v; p.seg_cap_a = c->seg_cap_a;
  p.causal = g.causal;
  p.stride_v = g.sim_stride_v; p.stride_a = g.sim_stride_a;
  p.scale = c->scale;
  p.scale_log2e = (float)((double)c->scale * 1.4426950408889634);
  p.lambda = g.lambda;
  p.shared_heads = g.select_scope == 1;
  p.d_model = g.sim_source == 2 ? g.d_model : 0;
  p.n_v = n_v; p.n = n; p.skip_budget = skip_budget;
  return p;
}

int check_chunk(const omnimem_ctx* c, const omnimem_chunk* ch, bool need_q) {
  if (!ch) return OMNIMEM_INVALID_ARG;
  if (ch->Nn_v < 0 || ch->Nn_a < 0) return OMNIMEM_INVALID_ARG;
  if (ch->Nn_v > c->cfg.max_chunk_v || ch->Nn_a > c->cfg.max_chunk_a) return OMNIMEM_CAPACITY;
  if (ch->Nn_v + ch->Nn_a > 0 && (!ch->k || !ch->v || (need_q && !ch->q))) return OMNIMEM_INVALID_ARG;
  return OMNIMEM_OK;
}
int check_cache(const omnimem_cache* ca) {
  return (ca && ca->k && ca->v && ca->n_v && ca->n) ? OMNIMEM_OK : OMNIMEM_INVALID_ARG;
}
// sim_source == 2 (R30): the hidden-state buffers must be there
int check_hidden(const omnimem_ctx* c, const omnimem_cache* ca, const omnimem_chunk* ch) {
  if (c->cfg.sim_source != 2) return OMNIMEM_OK;
  if (ca && !ca->h) return OMNIMEM_INVALID_ARG;
  if (ch && ch->Nn_v + ch->Nn_a > 0 && !ch->h) return OMNIMEM_INVALID_ARG;
  return OMNIMEM_OK;
}

struct StageTimer {
  omnimem_ctx* c;
  cudaStream_t st;
  int stage;
  StageTimer(omnimem_ctx* c_, cudaStream_t st_, int stage_) : c(c_), st(st_), stage(stage_) {
    if (c->profiling) { cudaEventRecord(c->ev[2 * stage], st); c->ev_used[stage] = true; }
  }
  ~StageTimer() { if (c->profiling) cudaEventRecord(c->ev[2 * stage + 1], st); }
};

void begin_call(omnimem_ctx* c) {
  c->launches = 0;
  for (int s = 0; s < OMNIMEM_N_STAGES; ++s) c->ev_used[s] = false;
}

// stages 1-3a on already validated arguments
int run_score(omnimem_ctx* c, const StepParams& p, StepBuffers& b, cudaStream_t st) {
  cudaError_t e;
  if (p.Nn > 0 && b.lse_in == nullptr) {
    StageTimer t(c, st, OMNIMEM_STAGE_LSE);
    e = c->use_tc ? launch_lse_tc(c, p, b, st, &c->launches) : launch_lse_simt(c, p, b, st, &c->launches);
    if (e != cudaSuccess) return fail_cuda(c, e);
  }
  {
    StageTimer t(c, st, OMNIMEM_STAGE_COLSUM);
    e = c->use_tc ? launch_colsum_tc(c, p, b, st, &c->launches) : launch_colsum_simt(c, p, b, st, &c->launches);
    if (e == cudaSuccess) e = launch_colsum_rescue(c, p, b, st, &c->launches);   // keys below fp32's range (R31)
    if (e != cudaSuccess) return fail_cuda(c, e);
  }
  {
    StageTimer t(c, st, OMNIMEM_STAGE_COSINE);
    e = launch_cosine(c, p, b, st, &c->launches);
    if (e != cudaSuccess) return fail_cuda(c, e);
  }
  {
    StageTimer t(c, st, OMNIMEM_STAGE_FINALIZE);
    e = launch_finalize(c, p, b, st, &c->launches);
    if (e != cudaSuccess) return fail_cuda(c, e);
  }
  return OMNIMEM_OK;
}

void fill_buffers(const omnimem_ctx* c, const omnimem_cache* src, const omnimem_chunk* ch, const omnimem_scores* out,
                  uint8_t* ws, const WsLayout& w, StepBuffers& b) {
  b.cacheK = src->k; b.cacheV = src->v; b.chunkK = ch->k; b.chunkV = ch->v; b.Q = ch->q;
  b.cacheH = src->h; b.chunkH = ch->h;
  b.lse_in = ch->lse;
  b.lse_out = out ? out->lse_out : nullptr;
  b.lse = ch->lse ? const_cast<float*>(ch->lse) : (b.lse_out ? b.lse_out : (float*)(ws + w.lse));
  b.lse2 = (float*)(ws + w.lse);
  b.row_entropy = out ? out->row_entropy : nullptr;
  b.a_v = out ? out->a_v : (float*)(ws + w.a_v);
  b.a_a = out ? out->a_a : (float*)(ws + w.a_a);
  b.s_v = out ? out->s_v : (float*)(ws + w.s_v);
  b.s_a = out ? out->s_a : (float*)(ws + w.s_a);
  b.psi_v = out ? out->psi_v : (float*)(ws + w.psi_v);
  b.psi_a = out ? out->psi_a : (float*)(ws + w.psi_a);
  b.la_v = (float*)(ws + w.la_v);
  b.la_a = (float*)(ws + w.la_a);
  b.rescue_items = (int32_t*)(ws + w.rescue_items);
  b.cosn = (float*)(ws + w.cosn);
  b.partials = (double*)(ws + w.partials);
  b.stats = out ? out->stats : (double*)(ws + w.stats);
}

int check_scores(const omnimem_scores* o) {
  return (o->a_v && o->a_a && o->s_v && o->s_a && o->psi_v && o->psi_a && o->stats) ? OMNIMEM_OK : OMNIMEM_INVALID_ARG;
}

// Time-interleaved chunk (R25'): derive the row <-> segment maps on the stream and hang them on the step parameters.
int set_chunk_maps(omnimem_ctx* c, const omnimem_chunk* ch, StepParams& p, cudaStream_t st) {
  p.row_of_seg = nullptr;
  p.seg_of_row = nullptr;
  if (!ch->modality || p.Nn == 0) return OMNIMEM_OK;
  int32_t* row_of_seg = c->chunk_maps;
  int32_t* seg_of_row = c->chunk_maps + (c->cfg.max_chunk_v + c->cfg.max_chunk_a);
  cudaError_t e = launch_chunk_maps(ch->modality, p.Nn, p.Nn_v, row_of_seg, seg_of_row, st, &c->launches);
  if (e != cudaSuccess) return fail_cuda(c, e);
  p.row_of_seg = row_of_seg;
  p.seg_of_row = seg_of_row;
  return OMNIMEM_OK;
}

int check_fused_args(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, const int32_t* layer_budget,
                     omnimem_cache* dst, omnimem_scores* opt_out, void* ws, size_t ws_bytes) {
  if (!ctx || !layer_budget || !ws) return OMNIMEM_INVALID_ARG;
  int rc = check_cache(src);
  if (rc) return rc;
  rc = check_cache(dst);
  if (rc) return rc;
  rc = check_chunk(ctx, chunk, true);
  if (rc) return rc;
  if (opt_out && (rc = check_scores(opt_out))) return rc;
  if (dst->k == src->k || dst->v == src->v || dst->n == src->n || dst->n_v == src->n_v) return OMNIMEM_INVALID_ARG;
  if ((rc = check_hidden(ctx, src, chunk)) || (rc = check_hidden(ctx, dst, nullptr))) return rc;
  if (ctx->cfg.sim_source == 2 && dst->h == src->h) return OMNIMEM_INVALID_ARG;
  if (ws_bytes < ws_layout(ctx).total) return OMNIMEM_WORKSPACE_TOO_SMALL;
  return OMNIMEM_OK;
}

// The fused step on layers [l0, l0 + Lg).  Every buffer of the step is laid out [L, ...] with the layer outermost and
// no stage looks across layers (the per-layer totals of Eq.14 are an input here, R21), so a layer range is the same
// problem with every per-layer pointer advanced by l0 and L = Lg.  Arguments are already validated.
int compress_layers(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, const int32_t* layer_budget,
                    omnimem_cache* dst, omnimem_scores* opt_out, int32_t* opt_idx_v, int32_t* opt_idx_a,
                    int32_t* opt_M_v, int32_t* opt_M_a, uint8_t* wsb, int l0, int Lg, cudaStream_t st) {
  const omnimem_config& g = ctx->cfg;
  const WsLayout w = ws_layout(ctx);
  const size_t es = g.dtype == OMNIMEM_FP32 ? 4 : 2;
  const size_t Nn = (size_t)chunk->Nn_v + chunk->Nn_a, Hq = g.n_q_heads, Hkv = g.n_kv_heads, D = g.head_dim;
  const size_t lz = (size_t)l0;
  auto adv = [](const void* p, size_t bytes) { return p ? (void*)((uint8_t*)const_cast<void*>(p) + bytes) : nullptr; };
  const size_t cache_b = lz * Hkv * g.cache_cap * D * es, kv_b = lz * Hkv * Nn * D * es, q_b = lz * Hq * Nn * D * es;
  const size_t segv_b = lz * Hkv * ctx->seg_cap_v * sizeof(float), sega_b = lz * Hkv * ctx->seg_cap_a * sizeof(float);
  const size_t row_b = lz * Hq * Nn * sizeof(float), idx_b = lz * Hkv * g.cache_cap * sizeof(int32_t);
  const size_t hc_b = lz * g.cache_cap * (size_t)g.d_model * es, hn_b = lz * Nn * (size_t)g.d_model * es;
  omnimem_cache s2{adv(src->k, cache_b), adv(src->v, cache_b), src->n_v + l0, src->n + l0, adv(src->h, hc_b)};
  omnimem_cache d2{adv(dst->k, cache_b), adv(dst->v, cache_b), dst->n_v + l0, dst->n + l0, adv(dst->h, hc_b)};
  omnimem_chunk c2 = *chunk;
  c2.k = adv(chunk->k, kv_b); c2.v = adv(chunk->v, kv_b); c2.q = adv(chunk->q, q_b); c2.h = adv(chunk->h, hn_b);
  c2.lse = (const float*)adv(chunk->lse, row_b);
  omnimem_scores o2{};
  if (opt_out) {
    o2.a_v = (float*)adv(opt_out->a_v, segv_b); o2.a_a = (float*)adv(opt_out->a_a, sega_b);
    o2.s_v = (float*)adv(opt_out->s_v, segv_b); o2.s_a = (float*)adv(opt_out->s_a, sega_b);
    o2.psi_v = (float*)adv(opt_out->psi_v, segv_b); o2.psi_a = (float*)adv(opt_out->psi_a, sega_b);
    o2.lse_out = (float*)adv(opt_out->lse_out, row_b); o2.row_entropy = (float*)adv(opt_out->row_entropy, row_b);
    o2.stats = opt_out->stats + lz * 8;
  }
  // the workspace regions are [L, per-layer bytes] too
  WsLayout w2 = w;
  const size_t lse_stride = ((Nn + 127) / 128) * 128;   // the row stride the scoring kernels use for this chunk
  w2.lse += lz * Hq * lse_stride * sizeof(float);
  w2.cosn += lz * Hkv * ((size_t)ctx->seg_cap_v + ctx->seg_cap_a) * sizeof(float);
  w2.partials += lz * 2 * (size_t)ctx->fin_blocks * 3 * sizeof(double);
  w2.a_v += segv_b; w2.la_v += segv_b; w2.s_v += segv_b; w2.psi_v += segv_b;
  w2.a_a += sega_b; w2.la_a += sega_b; w2.s_a += sega_b; w2.psi_a += sega_b;
  w2.stats += lz * 8 * sizeof(double);
  w2.M_v += lz * sizeof(int32_t); w2.M_a += lz * sizeof(int32_t);
  w2.idx_v += idx_b; w2.idx_a += idx_b;
  const int32_t* budget = layer_budget + l0;
  // layers with nothing to evict skip scoring unless the caller asked for the scores
  StepParams p = make_params(ctx, chunk->Nn_v, chunk->Nn_a, s2.n_v, s2.n, opt_out ? nullptr : budget, Lg);
  int rc = set_chunk_maps(ctx, chunk, p, st);
  if (rc) return rc;
  StepBuffers b{};
  fill_buffers(ctx, &s2, &c2, opt_out ? &o2 : nullptr, wsb, w2, b);
  rc = run_score(ctx, p, b, st);
  if (rc) return rc;
  int32_t* M_v = opt_M_v ? opt_M_v + l0 : (int32_t*)(wsb + w2.M_v);
  int32_t* M_a = opt_M_a ? opt_M_a + l0 : (int32_t*)(wsb + w2.M_a);
  int32_t* idx_v = opt_idx_v ? (int32_t*)adv(opt_idx_v, idx_b) : (int32_t*)(wsb + w2.idx_v);
  int32_t* idx_a = opt_idx_a ? (int32_t*)adv(opt_idx_a, idx_b) : (int32_t*)(wsb + w2.idx_a);
  cudaError_t e;
  {
    StageTimer t(ctx, st, OMNIMEM_STAGE_ALLOCATE);
    e = launch_allocate(ctx, p, b.stats, budget, 0, M_v, M_a, nullptr, st, &ctx->launches);
    if (e != cudaSuccess) return fail_cuda(ctx, e);
  }
  {
    StageTimer t(ctx, st, OMNIMEM_STAGE_SELECT);
    e = launch_select(ctx, p, b.psi_v, b.psi_a, M_v, M_a, idx_v, idx_a, st, &ctx->launches);
    if (e != cudaSuccess) return fail_cuda(ctx, e);
  }
  {
    StageTimer t(ctx, st, OMNIMEM_STAGE_COMPACT);
    e = launch_compact(ctx, p, s2.k, s2.v, c2.k, c2.v, idx_v, idx_a, M_v, M_a, d2.k, d2.v, d2.n_v, d2.n, st,
                       &ctx->launches);
    if (e == cudaSuccess && p.d_model > 0)
      e = launch_compact_hidden(ctx, p, s2.h, c2.h, idx_v, idx_a, M_v, M_a, d2.h, st, &ctx->launches);
    if (e != cudaSuccess) return fail_cuda(ctx, e);
  }
  return OMNIMEM_OK;
}

}  // namespace

extern "C" {

const char* omnimem_strerror(int status) {
  switch (status) {
    case OMNIMEM_OK: return "ok";
    case OMNIMEM_INVALID_ARG: return "invalid argument";
    case OMNIMEM_UNSUPPORTED: return "unsupported dtype, head_dim or device (needs sm_100)";
    case OMNIMEM_WORKSPACE_TOO_SMALL: return "workspace too small (see omnimem_workspace_bytes)";
    case OMNIMEM_CUDA_ERROR: return "CUDA error (see omnimem_last_cuda_error)";
    case OMNIMEM_CAPACITY: return "chunk exceeds the context capacities (max_chunk_v / max_chunk_a)";
    case OMNIMEM_STATIC_SCRATCH_EXCEEDED:
      return "omnimem_redundancy_static: n_layers * n_kv_heads * (2 * cache_cap + max_chunk_v + max_chunk_a) exceeds the "
             "built-in scratch array (OMNIMEM_STATIC_SCRATCH_FLOATS = 2^20 floats); call it per group of layers";
    default: return "unknown status";
  }
}

int omnimem_create(const omnimem_config* cfg, omnimem_ctx** out) {
  if (!cfg || !out) return OMNIMEM_INVALID_ARG;
  const omnimem_config& g = *cfg;
  if (g.n_layers <= 0 || g.n_q_heads <= 0 || g.n_kv_heads <= 0 || g.cache_cap <= 0 || g.max_chunk_v < 0 ||
      g.max_chunk_a < 0 || g.n_q_heads % g.n_kv_heads != 0 || g.sim_stride_v < 1 || g.sim_stride_a < 1 ||
      g.softmax_scale < 0.f || g.lambda < 0.f || g.ratio_r <= 0.f || g.temperature <= 0.f || g.budget_min < 0 ||
      g.budget_max < g.budget_min || g.sim_source < 0 || g.sim_source > 2 || (g.select_scope != 0 && g.select_scope != 1) || g.d_model < 0 || g.score_ctas < 0 ||
      (g.sim_source == 2 && (g.d_model == 0 || g.select_scope != 1 || (g.d_model * (g.dtype == OMNIMEM_FP32 ? 4 : 2)) % 16 != 0)) || g.n_kv_heads > 65535)
    return OMNIMEM_INVALID_ARG;
  if (g.dtype != OMNIMEM_FP32 && g.dtype != OMNIMEM_BF16) return OMNIMEM_UNSUPPORTED;
  if (g.head_dim != 64 && g.head_dim != 128) return OMNIMEM_UNSUPPORTED;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return OMNIMEM_CUDA_ERROR;
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) return OMNIMEM_CUDA_ERROR;
  if (prop.major != 10) return OMNIMEM_UNSUPPORTED;  // no fallback: this library is sm_100a code only
  omnimem_ctx* c = new (std::nothrow) omnimem_ctx();
  if (!c) return OMNIMEM_INVALID_ARG;
  c->cfg = g;
  c->device = dev;
  c->sm_count = prop.multiProcessorCount;
  c->cc_major = prop.major;
  c->cc_minor = prop.minor;
  c->seg_cap_v = g.cache_cap + g.max_chunk_v;
  c->seg_cap_a = g.cache_cap + g.max_chunk_a;
  const int mx = c->seg_cap_v > c->seg_cap_a ? c->seg_cap_v : c->seg_cap_a;
  c->fin_blocks = (mx + 255) / 256;
  c->scale = g.softmax_scale > 0.f ? g.softmax_scale : (float)(1.0 / sqrt((double)g.head_dim));
  c->use_tc = g.dtype == OMNIMEM_BF16 && g.head_dim == 128 && g.score_path == 0;
  c->last_err = cudaSuccess;
  c->profiling = false;
  c->launches = 0;
  c->encode_tiled = nullptr;
  for (int i = 0; i < 2 * OMNIMEM_N_STAGES; ++i) {
    e = cudaEventCreate(&c->ev[i]);
    if (e != cudaSuccess) { delete c; return OMNIMEM_CUDA_ERROR; }
  }
  for (int s = 0; s < OMNIMEM_N_STAGES; ++s) c->ev_used[s] = false;
  c->chunk_maps = nullptr;
  c->sched = nullptr;
  c->copy_stream = nullptr;
  for (int i = 0; i <= OMNIMEM_HOST_GROUPS; ++i) c->ev_copy[i] = nullptr;
  e = cudaMalloc((void**)&c->sched, 4 * sizeof(int32_t));
  if (e != cudaSuccess) { omnimem_destroy(c); return OMNIMEM_CUDA_ERROR; }
  if (g.max_chunk_v + g.max_chunk_a > 0) {
    e = cudaMalloc((void**)&c->chunk_maps, 2 * sizeof(int32_t) * ((size_t)g.max_chunk_v + g.max_chunk_a));
    if (e != cudaSuccess) { omnimem_destroy(c); return OMNIMEM_CUDA_ERROR; }
  }
  c->copy_stream = nullptr;
  for (int i = 0; i <= OMNIMEM_HOST_GROUPS; ++i) c->ev_copy[i] = nullptr;
  e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
  for (int i = 0; i <= OMNIMEM_HOST_GROUPS && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&c->ev_copy[i], cudaEventDisableTiming);
  if (e != cudaSuccess) { omnimem_destroy(c); return OMNIMEM_CUDA_ERROR; }
  *out = c;
  return OMNIMEM_OK;
}

int omnimem_destroy(omnimem_ctx* ctx) {
  if (!ctx) return OMNIMEM_INVALID_ARG;
  for (int i = 0; i < 2 * OMNIMEM_N_STAGES; ++i) cudaEventDestroy(ctx->ev[i]);
  for (int i = 0; i <= OMNIMEM_HOST_GROUPS; ++i) if (ctx->ev_copy[i]) cudaEventDestroy(ctx->ev_copy[i]);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  if (ctx->chunk_maps) cudaFree(ctx->chunk_maps);
  if (ctx->sched) cudaFree(ctx->sched);
  delete ctx;
  return OMNIMEM_OK;
}

size_t omnimem_workspace_bytes(const omnimem_ctx* ctx) { return ctx ? ws_layout(ctx).total : 0; }

int32_t omnimem_seg_cap(const omnimem_ctx* ctx, int32_t modality) {
  if (!ctx) return 0;
  return modality == 0 ? ctx->seg_cap_v : ctx->seg_cap_a;
}

const char* omnimem_last_cuda_error(const omnimem_ctx* ctx) {
  return ctx ? cudaGetErrorString(ctx->last_err) : "no context";
}

int omnimem_set_profiling(omnimem_ctx* ctx, int32_t enabled) {
  if (!ctx) return OMNIMEM_INVALID_ARG;
  ctx->profiling = enabled != 0;
  return OMNIMEM_OK;
}

int omnimem_get_stage_ms(omnimem_ctx* ctx, float* out, int32_t* launches_out) {
  if (!ctx || !out) return OMNIMEM_INVALID_ARG;
  for (int s = 0; s < OMNIMEM_N_STAGES; ++s) {
    out[s] = 0.f;
    if (ctx->profiling && ctx->ev_used[s]) {
      cudaError_t e = cudaEventSynchronize(ctx->ev[2 * s + 1]);
      if (e == cudaSuccess) e = cudaEventElapsedTime(&out[s], ctx->ev[2 * s], ctx->ev[2 * s + 1]);
      if (e != cudaSuccess) return fail_cuda(ctx, e);
    }
  }
  if (launches_out) *launches_out = ctx->launches;
  return OMNIMEM_OK;
}

int omnimem_score(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, omnimem_scores* out, void* ws,
                  size_t ws_bytes, void* stream) {
  if (!ctx || !out || !ws) return OMNIMEM_INVALID_ARG;
  int rc = check_cache(src);
  if (rc) return rc;
  rc = check_chunk(ctx, chunk, true);
  if (rc) return rc;
  rc = check_scores(out);
  if (rc) return rc;
  rc = check_hidden(ctx, src, chunk);
  if (rc) return rc;
  const WsLayout w = ws_layout(ctx);
  if (ws_bytes < w.total) return OMNIMEM_WORKSPACE_TOO_SMALL;
  begin_call(ctx);
  StepParams p = make_params(ctx, chunk->Nn_v, chunk->Nn_a, src->n_v, src->n, nullptr);
  if ((rc = set_chunk_maps(ctx, chunk, p, (cudaStream_t)stream))) return rc;
  StepBuffers b{};
  fill_buffers(ctx, src, chunk, out, (uint8_t*)ws, w, b);
  return run_score(ctx, p, b, (cudaStream_t)stream);
}

int omnimem_attend(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, void* y, float* lse_out, void* ws,
                   size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;   // the forward needs no scratch: NULL / 0 are accepted (the arguments stay for ABI stability)
  if (!ctx || !y || !lse_out) return OMNIMEM_INVALID_ARG;
  int rc = check_cache(src);
  if (rc) return rc;
  rc = check_chunk(ctx, chunk, true);
  if (rc) return rc;
  begin_call(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  StepParams p = make_params(ctx, chunk->Nn_v, chunk->Nn_a, src->n_v, src->n, nullptr);
  StepBuffers b{};
  b.cacheK = src->k; b.cacheV = src->v; b.chunkK = chunk->k; b.chunkV = chunk->v; b.Q = chunk->q;
  StageTimer t(ctx, st, OMNIMEM_STAGE_ATTEND);
  cudaError_t e = ctx->use_tc ? launch_attend_tc(ctx, p, b, y, lse_out, st, &ctx->launches)
                              : launch_attend_simt(ctx, p, b, y, lse_out, st, &ctx->launches);
  return e == cudaSuccess ? OMNIMEM_OK : fail_cuda(ctx, e);
}

int omnimem_allocate(omnimem_ctx* ctx, const double* stats, const int32_t* n_v, const int32_t* n, int32_t Nn_v,
                     int32_t Nn_a, const int32_t* layer_budget, int64_t total_budget, int32_t* M_v, int32_t* M_a,
                     int32_t* layer_budget_out, void* stream) {
  if (!ctx || !stats || !n_v || !n || !M_v || !M_a || Nn_v < 0 || Nn_a < 0) return OMNIMEM_INVALID_ARG;
  if (!layer_budget && total_budget < 0) return OMNIMEM_INVALID_ARG;
  if (Nn_v > ctx->cfg.max_chunk_v || Nn_a > ctx->cfg.max_chunk_a) return OMNIMEM_CAPACITY;
  begin_call(ctx);
  StepParams p = make_params(ctx, Nn_v, Nn_a, n_v, n, nullptr);
  StageTimer t(ctx, (cudaStream_t)stream, OMNIMEM_STAGE_ALLOCATE);
  cudaError_t e = launch_allocate(ctx, p, stats, layer_budget, total_budget, M_v, M_a, layer_budget_out,
                                  (cudaStream_t)stream, &ctx->launches);
  return e == cudaSuccess ? OMNIMEM_OK : fail_cuda(ctx, e);
}

int omnimem_calibrate_accumulate(omnimem_ctx* ctx, const double* stats, double* acc, void* stream) {
  if (!ctx || !stats || !acc) return OMNIMEM_INVALID_ARG;
  begin_call(ctx);
  cudaError_t e = launch_calib_accumulate(ctx->cfg.n_layers, stats, acc, (cudaStream_t)stream, &ctx->launches);
  return e == cudaSuccess ? OMNIMEM_OK : fail_cuda(ctx, e);
}

int omnimem_calibrate_budgets(omnimem_ctx* ctx, const double* acc, int64_t total_budget, double* mean_stats_out,
                              int32_t* layer_budget_out, void* stream) {
  if (!ctx || !acc || !mean_stats_out || !layer_budget_out || total_budget < 0) return OMNIMEM_INVALID_ARG;
  begin_call(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = launch_calib_mean(ctx->cfg.n_layers, acc, mean_stats_out, st, &ctx->launches);
  if (e != cudaSuccess) return fail_cuda(ctx, e);
  StepParams p = make_params(ctx, 0, 0, nullptr, nullptr, nullptr);
  e = launch_allocate(ctx, p, mean_stats_out, nullptr, total_budget, nullptr, nullptr, layer_budget_out, st, &ctx->launches);
  return e == cudaSuccess ? OMNIMEM_OK : fail_cuda(ctx, e);
}

int omnimem_select(omnimem_ctx* ctx, const float* psi_v, const float* psi_a, const int32_t* n_v, const int32_t* n,
                   int32_t Nn_v, int32_t Nn_a, const int32_t* M_v, const int32_t* M_a, int32_t* idx_v, int32_t* idx_a,
                   void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (!ctx || !psi_v || !psi_a || !n_v || !n || !M_v || !M_a || !idx_v || !idx_a || Nn_v < 0 || Nn_a < 0)
    return OMNIMEM_INVALID_ARG;
  if (Nn_v > ctx->cfg.max_chunk_v || Nn_a > ctx->cfg.max_chunk_a) return OMNIMEM_CAPACITY;
  begin_call(ctx);
  StepParams p = make_params(ctx, Nn_v, Nn_a, n_v, n, nullptr);
  StageTimer t(ctx, (cudaStream_t)stream, OMNIMEM_STAGE_SELECT);
  cudaError_t e = launch_select(ctx, p, psi_v, psi_a, M_v, M_a, idx_v, idx_a, (cudaStream_t)stream, &ctx->launches);
  return e == cudaSuccess ? OMNIMEM_OK : fail_cuda(ctx, e);
}

int omnimem_compact(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk, const int32_t* idx_v,
                    const int32_t* idx_a, const int32_t* M_v, const int32_t* M_a, omnimem_cache* dst, void* stream) {
  if (!ctx || !idx_v || !idx_a || !M_v || !M_a) return OMNIMEM_INVALID_ARG;
  int rc = check_cache(src);
  if (rc) return rc;
  rc = check_cache(dst);
  if (rc) return rc;
  rc = check_chunk(ctx, chunk, false);
  if (rc) return rc;
  if (dst->k == src->k || dst->v == src->v || dst->n == src->n || dst->n_v == src->n_v) return OMNIMEM_INVALID_ARG;
  if ((rc = check_hidden(ctx, src, chunk)) || (rc = check_hidden(ctx, dst, nullptr))) return rc;
  begin_call(ctx);
  StepParams p = make_params(ctx, chunk->Nn_v, chunk->Nn_a, src->n_v, src->n, nullptr);
  if ((rc = set_chunk_maps(ctx, chunk, p, (cudaStream_t)stream))) return rc;
  StageTimer t(ctx, (cudaStream_t)stream, OMNIMEM_STAGE_COMPACT);
  cudaError_t e = launch_compact(ctx, p, src->k, src->v, chunk->k, chunk->v, idx_v, idx_a, M_v, M_a, dst->k, dst->v,
                                 dst->n_v, dst->n, (cudaStream_t)stream, &ctx->launches);
  if (e == cudaSuccess && p.d_model > 0)   // the retained hidden states follow the kept tokens (R30)
    e = launch_compact_hidden(ctx, p, src->h, chunk->h, idx_v, idx_a, M_v, M_a, dst->h, (cudaStream_t)stream, &ctx->launches);
  return e == cudaSuccess ? OMNIMEM_OK : fail_cuda(ctx, e);
}

int omnimem_compress_chunk(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* chunk,
                           const int32_t* layer_budget, omnimem_cache* dst, omnimem_scores* opt_out, int32_t* opt_idx_v,
                           int32_t* opt_idx_a, int32_t* opt_M_v, int32_t* opt_M_a, void* ws, size_t ws_bytes,
                           void* stream) {
  int rc = check_fused_args(ctx, src, chunk, layer_budget, dst, opt_out, ws, ws_bytes);
  if (rc) return rc;
  begin_call(ctx);
  return compress_layers(ctx, src, chunk, layer_budget, dst, opt_out, opt_idx_v, opt_idx_a, opt_M_v, opt_M_a,
                         (uint8_t*)ws, 0, ctx->cfg.n_layers, (cudaStream_t)stream);
}

int omnimem_compress_chunk_host(omnimem_ctx* ctx, const omnimem_cache* src, const omnimem_chunk* host_chunk,
                                const omnimem_chunk* dev_chunk, const int32_t* layer_budget, omnimem_cache* dst,
                                int32_t* host_M_v, int32_t* host_M_a, int64_t* h2d_bytes, int64_t* d2h_bytes, void* ws,
                                size_t ws_bytes, void* stream) {
  if (!ctx || !host_chunk || !dev_chunk || !host_M_v || !host_M_a || !ws) return OMNIMEM_INVALID_ARG;
  int rc = check_chunk(ctx, host_chunk, true);
  if (rc) return rc;
  if (!dev_chunk->k || !dev_chunk->v || !dev_chunk->q || (host_chunk->lse && !dev_chunk->lse)) return OMNIMEM_INVALID_ARG;
  if (ctx->cfg.sim_source == 2 && (!host_chunk->h || !dev_chunk->h)) return OMNIMEM_INVALID_ARG;
  if (host_chunk->modality && host_chunk->Nn_v + host_chunk->Nn_a > 0 && !dev_chunk->modality) return OMNIMEM_INVALID_ARG;
  omnimem_chunk ch = *dev_chunk;
  ch.Nn_v = host_chunk->Nn_v;
  ch.Nn_a = host_chunk->Nn_a;
  if (!host_chunk->lse) ch.lse = nullptr;
  if (!host_chunk->modality) ch.modality = nullptr;
  rc = check_fused_args(ctx, src, &ch, layer_budget, dst, nullptr, ws, ws_bytes);
  if (rc) return rc;
  const WsLayout w = ws_layout(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  const omnimem_config& g = ctx->cfg;
  const int L = g.n_layers;
  const size_t es = g.dtype == OMNIMEM_FP32 ? 4 : 2;
  const size_t Nn = (size_t)host_chunk->Nn_v + host_chunk->Nn_a;
  const size_t kv_layer = (size_t)g.n_kv_heads * Nn * g.head_dim * es;      // bytes per layer
  const size_t q_layer = (size_t)g.n_q_heads * Nn * g.head_dim * es;
  const size_t lse_layer = host_chunk->lse ? (size_t)g.n_q_heads * Nn * sizeof(float) : 0;
  const size_t h_layer = g.sim_source == 2 ? Nn * (size_t)g.d_model * es : 0;
  uint8_t* wsb = (uint8_t*)ws;
  begin_call(ctx);
  // Layers are independent through the whole step, so the chunk is copied and compressed in groups of layers: the
  // copy of group g + 1 (on the context's copy stream) overlaps the kernels of group g (on `stream`).
  // Group sizes grow geometrically (1, 2, 3, 4, 6, 9, ... layers): only the first, one-layer copy is exposed, each later
  // copy is shorter than the kernels it hides behind (a layer computes for longer than it copies), and the big late
  // groups keep the scoring kernels' tail waves few.  The last of the OMNIMEM_HOST_GROUPS groups takes the rest.
  int group_size[OMNIMEM_HOST_GROUPS];
  int n_groups = 0;
  for (int left = L, sz = 1; left > 0; ++n_groups) {
    const int take = (n_groups == OMNIMEM_HOST_GROUPS - 1 || sz > left) ? left : sz;
    group_size[n_groups] = take;
    left -= take;
    sz = sz + 1 > sz * 3 / 2 ? sz + 1 : sz * 3 / 2;
  }
  cudaError_t e = cudaEventRecord(ctx->ev_copy[OMNIMEM_HOST_GROUPS], st);   // staging buffers are free once `stream` got here
  if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_copy[OMNIMEM_HOST_GROUPS], 0);
  if (e != cudaSuccess) return fail_cuda(ctx, e);
  auto at = [](const void* p, size_t bytes) { return (void*)((uint8_t*)const_cast<void*>(p) + bytes); };
  // an error after this point leaves copies in flight that read the caller's host buffers: wait for them before returning
  auto fail_mid = [&](int status) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamSynchronize(st); return status; };
  if (host_chunk->modality && Nn > 0) {   // HOST [Nn] -> the device staging copy, ahead of the first group
    e = cudaMemcpyAsync(const_cast<int32_t*>(dev_chunk->modality), host_chunk->modality, Nn * sizeof(int32_t),
                        cudaMemcpyHostToDevice, ctx->copy_stream);
    if (e != cudaSuccess) return fail_mid(fail_cuda(ctx, e));
  }
  int gi = 0;
  for (int l0 = 0; gi < n_groups; l0 += group_size[gi], ++gi) {
    const int Lg = group_size[gi];
    if (Nn > 0) {
      cudaStream_t cs = ctx->copy_stream;
      e = cudaMemcpyAsync(at(dev_chunk->k, l0 * kv_layer), at(host_chunk->k, l0 * kv_layer), Lg * kv_layer, cudaMemcpyHostToDevice, cs);
      if (e == cudaSuccess)
        e = cudaMemcpyAsync(at(dev_chunk->q, l0 * q_layer), at(host_chunk->q, l0 * q_layer), Lg * q_layer, cudaMemcpyHostToDevice, cs);
      if (e == cudaSuccess && lse_layer)
        e = cudaMemcpyAsync(at(dev_chunk->lse, l0 * lse_layer), at(host_chunk->lse, l0 * lse_layer), Lg * lse_layer, cudaMemcpyHostToDevice, cs);
      if (e == cudaSuccess)
        e = cudaMemcpyAsync(at(dev_chunk->v, l0 * kv_layer), at(host_chunk->v, l0 * kv_layer), Lg * kv_layer, cudaMemcpyHostToDevice, cs);
      if (e == cudaSuccess && h_layer)
        e = cudaMemcpyAsync(at(dev_chunk->h, l0 * h_layer), at(host_chunk->h, l0 * h_layer), Lg * h_layer, cudaMemcpyHostToDevice, cs);
      if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_copy[gi], cs);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ctx->ev_copy[gi], 0);
      if (e != cudaSuccess) return fail_mid(fail_cuda(ctx, e));
    }
    rc = compress_layers(ctx, src, &ch, layer_budget, dst, nullptr, nullptr, nullptr, nullptr, nullptr, wsb, l0, Lg, st);
    if (rc) return fail_mid(rc);
  }
  const size_t mb = (size_t)L * sizeof(int32_t);
  e = cudaMemcpyAsync(host_M_v, wsb + w.M_v, mb, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(host_M_a, wsb + w.M_a, mb, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail_mid(fail_cuda(ctx, e));
  if (h2d_bytes) *h2d_bytes = (int64_t)(Nn > 0 ? (size_t)L * (2 * kv_layer + q_layer + lse_layer + h_layer) : 0);
  if (d2h_bytes) *d2h_bytes = (int64_t)(2 * mb);
  return OMNIMEM_OK;
}

}  // extern "C"
