/*
 * oracle/omnimem_ref.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what one OmniMem per-chunk KV-cache
 * compression step computes (arxiv/paper_2606_07577, section 3,
 * Eq.1-14).  It exists so that the CUDA path can be checked against something
 * that a reader can compare with the paper by eye.  It shares no code, header,
 * table or helper with the CUDA path under paper_2606_07577_b200/csrc, and
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * Citations "P:<n>" are line numbers of /root/reference/PAPER.md; "R<k>" are
 * the readings of the paper listed in DESIGN.md (section "Readings").
 *
 * Every floating-point quantity is a C double.  The caller converts the
 * (already bf16- or fp32-rounded) inputs to double exactly, so the oracle sees
 * the very values the GPU sees.  The only non-double outputs are psi (rounded
 * once to float: the public score array that selection consumes, R13) and the
 * compacted caches (raw bytes, moved not computed).
 *
 * Loops follow the paper's order: attention rows -> column sums (Eq.6),
 * adjacent cosine (Eq.7), psi (Eq.8), AVBA statistics (Eq.9-10, 13), split
 * (Eq.11-12), layer totals (Eq.14), top-M (Eq.4-5), prune.  No tiling, no
 * fusion.  OpenMP only distributes independent query rows over threads
 * (declarative `reduction`, no hand-written blocking).
 *
 * Pins (tests/test_oracle_pins.py) -- each function below is checked against
 * something other than itself.  omnimem_ref_layer_budgets (Eq.14 + clamp and
 * rounding, R20) is pinned by the water-filling form the mathematics fixes,
 * b_l = clip(kappa pi_l, B_min, B_max) with sum_l b_l = total, found by plain
 * bisection in numpy on 240 seeded cases, plus a numpy largest-remainder
 * integerisation and two closed forms.  What stays unpinned is only the
 * end-to-end numeric output as a whole: the paper prints no worked example.
 */
#define _GNU_SOURCE /* qsort_r */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int32_t L, Hq, Hkv, D;
  int32_t cache_cap;        /* rows per (layer, kv head) in the cache buffers (row stride)  */
  int32_t Nn_v, Nn_a;       /* chunk rows: visual block [0,Nn_v) then audio block           */
  int32_t causal;           /* R3: 1 = chunk key t visible to chunk query i iff t <= i      */
  int32_t sim_stride_v;     /* R11: neighbour distance of Eq.7 per modality (1 = literal)   */
  int32_t sim_stride_a;
  int32_t seg_cap_v;        /* row stride of the per-modality output arrays                 */
  int32_t seg_cap_a;
  double scale;             /* R4: softmax scale c (caller passes 1/sqrt(D))                */
  double lambda;            /* Eq.8  (default 0.02 P:159)                            */
  double ratio_r;           /* Eq.11-12 prior visual:audio ratio r (default 5)       */
  double temperature;       /* Eq.14 T (default 0.2 P:159)                           */
  int64_t budget_min;       /* Eq.14 clamp [B_min, B_max]; 0,0 = no clamp           */
  int64_t budget_max;
  const int32_t* chunk_modality; /* R25': NULL = modality-blocked chunk (visual block then audio block); else
                                    [Nn] with 0 = visual, 1 = audio for each chunk row in TRUE temporal order
                                    (time-interleaved chunk, "a specific number of audio and visual tokens") */
} omnimem_ref_params;

#define IDX3(a, b, c, B, C) ((((int64_t)(a)) * (B) + (b)) * (int64_t)(C) + (c))

/* ---- O1: logical sequences (Eq.2-3) ------------------------------------------
 * Key order seen by attention (R2: ONE joint softmax): cached visual, cached audio,
 * then the chunk's rows in storage order (new visual, new audio when blocked; true temporal
 * order when chunk_modality is given; the causal mask of R3 follows that order).  Row k: */
static const double* key_row(const omnimem_ref_params* p, const double* cacheX, const double* chunkX,
                             int l, int h, int Nc, int k) {
  const int Nn = p->Nn_v + p->Nn_a;
  if (k < Nc) return cacheX + IDX3(l * p->Hkv + h, k, 0, p->cache_cap, p->D);
  return chunkX + IDX3(l * p->Hkv + h, k - Nc, 0, Nn, p->D);
}

/* Per-modality appended sequence K~_m = [cache_m ; chunk_m] (Eq.3).  Segment-local index t of
 * modality m (0 = visual, 1 = audio) -> index in the logical sequence above. */
static int seg_to_logical(const omnimem_ref_params* p, int n_v, int n, int m, int t) {
  const int n_m = m == 0 ? n_v : n - n_v;
  if (t < n_m) return m == 0 ? t : n_v + t;                  /* cached rows: visual block, then audio block  */
  if (p->chunk_modality == NULL)                             /* blocked chunk (R25)                          */
    return m == 0 ? n + (t - n_v) : n + p->Nn_v + (t - n_m);
  int want = t - n_m;                                        /* interleaved chunk: the want-th row of modality m */
  for (int r = 0; r < p->Nn_v + p->Nn_a; ++r)
    if (p->chunk_modality[r] == m && want-- == 0) return n + r;
  return -1;                                                 /* Nn_v / Nn_a do not match the map             */
}
static int seg_len(const omnimem_ref_params* p, int n_v, int n, int m) {
  return m == 0 ? n_v + p->Nn_v : (n - n_v) + p->Nn_a;
}

/* ---- O2: attention of the chunk's queries + importance (Eq.1 softmax, Eq.6) ----
 * For KV head h, query heads j = h*G+g (standard GQA mapping), query i:
 *   z_k = c <q_i, k_k>  over visible k;  p_k = softmax(z)_k;  a[l,h,k] += p_k   (R5: G heads summed)
 *   lse[l,j,i] = log sum_k exp(z_k);  rowH[l,j,i] = -sum_k p_k log p_k (diagnostic, R16).
 * a_log is [L,Hkv,cache_cap+Nn] in LOGICAL key order; entries >= n[l]+Nn are set to 0. */
int omnimem_ref_attention(const omnimem_ref_params* p, const double* cacheK, const int32_t* n,
                          const double* chunkK, const double* Q, double* a_log, double* lse, double* rowH) {
  const int Nn = p->Nn_v + p->Nn_a, G = p->Hq / p->Hkv, D = p->D;
  const int Nkcap = p->cache_cap + Nn;
  if (p->Hq % p->Hkv != 0) return -1;
  for (int l = 0; l < p->L; ++l) {
    for (int h = 0; h < p->Hkv; ++h) {
      const int Nc = n[l], Nk = Nc + Nn;
      double* acc = a_log + IDX3(l, h, 0, p->Hkv, Nkcap);
      for (int k = 0; k < Nkcap; ++k) acc[k] = 0.0;
      if (Nk == 0) continue;
#pragma omp parallel for reduction(+ : acc[:Nk]) schedule(dynamic, 4)
      for (int ri = 0; ri < G * Nn; ++ri) {
        const int g = ri / Nn, i = ri % Nn, j = h * G + g;
        const double* q = Q + IDX3(l * p->Hq + j, i, 0, Nn, D);
        const int nvis = p->causal ? Nc + i + 1 : Nk; /* R3 */
        double* z = (double*)malloc(sizeof(double) * (size_t)nvis);
        double m = -INFINITY;
        for (int k = 0; k < nvis; ++k) {
          const double* kr = key_row(p, cacheK, chunkK, l, h, Nc, k);
          double dot = 0.0;
#pragma omp simd reduction(+ : dot)
          for (int d = 0; d < D; ++d) dot += q[d] * kr[d];
          z[k] = p->scale * dot;
          if (z[k] > m) m = z[k];
        }
        double Z = 0.0;
        for (int k = 0; k < nvis; ++k) Z += exp(z[k] - m);
        double Hrow = 0.0;
        for (int k = 0; k < nvis; ++k) {
          const double pk = exp(z[k] - m) / Z;
          acc[k] += pk;
          if (pk > 0.0) Hrow -= pk * log(pk);
        }
        if (lse) lse[IDX3(l, j, i, p->Hq, Nn)] = m + log(Z);
        if (rowH) rowH[IDX3(l, j, i, p->Hq, Nn)] = Hrow;
        free(z);
      }
    }
  }
  return 0;
}

/* ---- A1: the chunk's multi-head self-attention over both caches and the chunk (Eq.1, Eq.2) ----
 * Y_c = MHSA(Q_c, K_c, V_c, O_c, P_c): for query head j = h*G+g and chunk query i,
 *   Y[l,j,i,:] = sum_{k visible} softmax_k(c <q_i, k_k>) v_k
 * over the same logical key sequence and the same mask as O2 (cached visual, cached audio, chunk rows in storage
 * order; causal inside the chunk, R2-R3); values V follow the keys' order.  lse[l,j,i] is the row's log-sum-exp,
 * the quantity score pass 2 needs (Eq.6).  absY (optional) = sum_k p_k |v_k|: the magnitude that bounds the rounding
 * error of an implementation that rounds p or Y to bf16.  Y, absY: [L,Hq,Nn,D]; lse: [L,Hq,Nn]. */
int omnimem_ref_mhsa(const omnimem_ref_params* p, const double* cacheK, const double* cacheV, const int32_t* n,
                     const double* chunkK, const double* chunkV, const double* Q, double* Y, double* lse,
                     double* absY) {
  const int Nn = p->Nn_v + p->Nn_a, G = p->Hq / p->Hkv, D = p->D;
  if (p->Hq % p->Hkv != 0) return -1;
  for (int l = 0; l < p->L; ++l) {
    const int Nc = n[l], Nk = Nc + Nn;
#pragma omp parallel for schedule(dynamic, 4)
    for (int ri = 0; ri < p->Hq * Nn; ++ri) {
      const int j = ri / Nn, i = ri % Nn, h = j / G;
      const double* q = Q + IDX3(l * p->Hq + j, i, 0, Nn, D);
      double* y = Y + IDX3(l * p->Hq + j, i, 0, Nn, D);
      double* ay = absY ? absY + IDX3(l * p->Hq + j, i, 0, Nn, D) : NULL;
      const int nvis = p->causal ? Nc + i + 1 : Nk; /* R3 */
      double* z = (double*)malloc(sizeof(double) * (size_t)(nvis > 0 ? nvis : 1));
      double m = -INFINITY;
      for (int k = 0; k < nvis; ++k) {
        const double* kr = key_row(p, cacheK, chunkK, l, h, Nc, k);
        double dot = 0.0;
        for (int d = 0; d < D; ++d) dot += q[d] * kr[d];
        z[k] = p->scale * dot;
        if (z[k] > m) m = z[k];
      }
      double Z = 0.0;
      for (int k = 0; k < nvis; ++k) Z += exp(z[k] - m);
      for (int d = 0; d < D; ++d) {
        y[d] = 0.0;
        if (ay) ay[d] = 0.0;
      }
      for (int k = 0; k < nvis; ++k) {
        const double pk = exp(z[k] - m) / Z;
        const double* vr = key_row(p, cacheV, chunkV, l, h, Nc, k);
        for (int d = 0; d < D; ++d) {
          y[d] += pk * vr[d];
          if (ay) ay[d] += pk * fabs(vr[d]);
        }
      }
      if (lse) lse[IDX3(l, j, i, p->Hq, Nn)] = m + log(Z);
      free(z);
    }
  }
  return 0;
}

/* Split a logical-order array into the two per-modality segment arrays [L,Hkv,seg_cap_m]. */
int omnimem_ref_split(const omnimem_ref_params* p, const double* a_log, const int32_t* n_v, const int32_t* n,
                      double* a_v, double* a_a) {
  const int Nn = p->Nn_v + p->Nn_a, Nkcap = p->cache_cap + Nn;
  for (int l = 0; l < p->L; ++l)
    for (int h = 0; h < p->Hkv; ++h)
      for (int m = 0; m < 2; ++m) {
        const int Km = seg_len(p, n_v[l], n[l], m);
        const int cap = m == 0 ? p->seg_cap_v : p->seg_cap_a;
        double* out = (m == 0 ? a_v : a_a) + IDX3(l, h, 0, p->Hkv, cap);
        if (Km > cap) return -5;
        for (int t = 0; t < Km; ++t)
          out[t] = a_log[IDX3(l, h, seg_to_logical(p, n_v[l], n[l], m, t), p->Hkv, Nkcap)];
        for (int t = Km; t < cap; ++t) out[t] = 0.0;
      }
  return 0;
}

/* ---- O3: redundancy (Eq.7; on value vectors per P:103, R8) ------------------------
 * s_t = [cos(x_t, x_{t+sigma}) + cos(x_{t-sigma}, x_t)] / 2 inside the modality's appended
 * sequence (R9); a missing neighbour is left out of the mean, none => 0 (R10);
 * cos = <x,y> / max(|x||y|, 1e-8), s clamped to [-1,1] (R12).  X is V (or K if the caller
 * passes K: sim_source, R8). */
static double cosine(const double* x, const double* y, int D) {
  double xy = 0.0, xx = 0.0, yy = 0.0;
  for (int d = 0; d < D; ++d) {
    xy += x[d] * y[d];
    xx += x[d] * x[d];
    yy += y[d] * y[d];
  }
  double den = sqrt(xx) * sqrt(yy);
  if (den < 1e-8) den = 1e-8;
  return xy / den;
}

int omnimem_ref_redundancy(const omnimem_ref_params* p, const double* cacheX, const int32_t* n_v,
                           const int32_t* n, const double* chunkX, double* s_v, double* s_a) {
  for (int l = 0; l < p->L; ++l)
    for (int h = 0; h < p->Hkv; ++h)
      for (int m = 0; m < 2; ++m) {
        const int Km = seg_len(p, n_v[l], n[l], m);
        const int cap = m == 0 ? p->seg_cap_v : p->seg_cap_a;
        const int sg = m == 0 ? p->sim_stride_v : p->sim_stride_a;
        double* out = (m == 0 ? s_v : s_a) + IDX3(l, h, 0, p->Hkv, cap);
        if (Km > cap || sg < 1) return -1;
#pragma omp parallel for schedule(static)
        for (int t = 0; t < Km; ++t) {
          const double* x = key_row(p, cacheX, chunkX, l, h, n[l], seg_to_logical(p, n_v[l], n[l], m, t));
          double sum = 0.0;
          int cnt = 0;
          if (t + sg < Km) {
            const double* y = key_row(p, cacheX, chunkX, l, h, n[l], seg_to_logical(p, n_v[l], n[l], m, t + sg));
            sum += cosine(x, y, p->D);
            ++cnt;
          }
          if (t - sg >= 0) {
            const double* y = key_row(p, cacheX, chunkX, l, h, n[l], seg_to_logical(p, n_v[l], n[l], m, t - sg));
            sum += cosine(y, x, p->D);
            ++cnt;
          }
          double s = cnt ? sum / cnt : 0.0;
          if (s > 1.0) s = 1.0;
          if (s < -1.0) s = -1.0;
          out[t] = s;
        }
        for (int t = Km; t < cap; ++t) out[t] = 0.0;
      }
  return 0;
}

/* ---- O4: selection score (Eq.8) --------------------------------------------------
 * psi = a^lambda (1 - s), C pow semantics (0^lambda = 0 for lambda > 0, x^0 = 1, R13); rounded ONCE
 * to float: the fp32 array is the public score that Select consumes. */
int omnimem_ref_psi(const omnimem_ref_params* p, const int32_t* n_v, const int32_t* n, const double* a_v,
                    const double* a_a, const double* s_v, const double* s_a, float* psi_v, float* psi_a) {
  for (int l = 0; l < p->L; ++l)
    for (int h = 0; h < p->Hkv; ++h)
      for (int m = 0; m < 2; ++m) {
        const int Km = seg_len(p, n_v[l], n[l], m);
        const int cap = m == 0 ? p->seg_cap_v : p->seg_cap_a;
        const double* a = (m == 0 ? a_v : a_a) + IDX3(l, h, 0, p->Hkv, cap);
        const double* s = (m == 0 ? s_v : s_a) + IDX3(l, h, 0, p->Hkv, cap);
        float* out = (m == 0 ? psi_v : psi_a) + IDX3(l, h, 0, p->Hkv, cap);
        for (int t = 0; t < Km; ++t) out[t] = (float)(pow(a[t], p->lambda) * (1.0 - s[t]));
        for (int t = Km; t < cap; ++t) out[t] = 0.0f;
      }
  return 0;
}

/* ---- O4': the paper-literal selection score, one per token and layer (R29) --------------------
 * Eq.4-5 write the index sets I_{c,v}^{(l)}, I_{c,a}^{(l)} with no head index and Eq.6 an
 * importance a_k with none either: the token is scored once per layer.  Reading R29: the importance is summed
 * over ALL query heads (= the sum over KV heads of the per-group sums), the redundancy of Eq.7 taken on value
 * rows is averaged over the KV heads, psi = A^lambda (1 - S) (Eq.8).  Every head's row of the output gets
 * the same score, so Select returns the same index set for every head of the layer. */
int omnimem_ref_psi_shared(const omnimem_ref_params* p, const int32_t* n_v, const int32_t* n, const double* a_v,
                           const double* a_a, const double* s_v, const double* s_a, float* psi_v, float* psi_a) {
  for (int l = 0; l < p->L; ++l)
    for (int m = 0; m < 2; ++m) {
      const int Km = seg_len(p, n_v[l], n[l], m);
      const int cap = m == 0 ? p->seg_cap_v : p->seg_cap_a;
      const double* a = m == 0 ? a_v : a_a;
      const double* s = m == 0 ? s_v : s_a;
      float* out = m == 0 ? psi_v : psi_a;
      for (int t = 0; t < cap; ++t) {
        double A = 0.0, S = 0.0;
        for (int h = 0; h < p->Hkv; ++h) {
          A += a[IDX3(l, h, t, p->Hkv, cap)];
          S += s[IDX3(l, h, t, p->Hkv, cap)];
        }
        const float v = t < Km ? (float)(pow(A, p->lambda) * (1.0 - S / p->Hkv)) : 0.0f;
        for (int h = 0; h < p->Hkv; ++h) out[IDX3(l, h, t, p->Hkv, cap)] = v;
      }
    }
  return 0;
}

/* ---- O5: AVBA statistics (Eq.9-10; Eq.13) -------------------------------
 * Per layer and modality: A_m[t] = sum_h a[l,h,m,t]; abar = A_m / sum_t A_m (R16);
 * Hn_m = H[abar] / ln K_m (natural log, 0 ln 0 = 0, K_m <= 1 or empty mass => 0, R15);
 * sbar_m = mean over heads and tokens of s (R17); C_m = Hn_m (1 - sbar_m).
 * Layer-wide (Eq.13, R18): the same over the union of both segments, normalised by ln(K_v+K_a).
 * stats[l] = {Hn_v, Hn_a, sbar_v, sbar_a, C_v, C_a, Hn_all, sbar_all}. */
int omnimem_ref_stats(const omnimem_ref_params* p, const int32_t* n_v, const int32_t* n, const double* a_v,
                      const double* a_a, const double* s_v, const double* s_a, double* stats) {
  for (int l = 0; l < p->L; ++l) {
    double Hn[2], sbar[2];
    const int Kv = seg_len(p, n_v[l], n[l], 0), Ka = seg_len(p, n_v[l], n[l], 1);
    double* A_all = (double*)malloc(sizeof(double) * (size_t)(Kv + Ka + 1));
    double s_sum_all = 0.0;
    for (int m = 0; m < 2; ++m) {
      const int Km = m == 0 ? Kv : Ka;
      const int cap = m == 0 ? p->seg_cap_v : p->seg_cap_a;
      double* A = A_all + (m == 0 ? 0 : Kv);
      double S = 0.0, s_sum = 0.0;
      for (int t = 0; t < Km; ++t) {
        A[t] = 0.0;
        for (int h = 0; h < p->Hkv; ++h) {
          A[t] += (m == 0 ? a_v : a_a)[IDX3(l, h, t, p->Hkv, cap)];
          s_sum += (m == 0 ? s_v : s_a)[IDX3(l, h, t, p->Hkv, cap)];
        }
        S += A[t];
      }
      double H = 0.0;
      if (S > 0.0)
        for (int t = 0; t < Km; ++t) {
          const double ab = A[t] / S;
          if (ab > 0.0) H -= ab * log(ab);
        }
      Hn[m] = (Km > 1 && S > 0.0) ? H / log((double)Km) : 0.0;
      sbar[m] = Km > 0 ? s_sum / ((double)Km * p->Hkv) : 0.0;
      s_sum_all += s_sum;
    }
    const int Kall = Kv + Ka;
    double S = 0.0, H = 0.0;
    for (int t = 0; t < Kall; ++t) S += A_all[t];
    if (S > 0.0)
      for (int t = 0; t < Kall; ++t) {
        const double ab = A_all[t] / S;
        if (ab > 0.0) H -= ab * log(ab);
      }
    double* st = stats + (int64_t)l * 8;
    st[0] = Hn[0];
    st[1] = Hn[1];
    st[2] = sbar[0];
    st[3] = sbar[1];
    st[4] = Hn[0] * (1.0 - sbar[0]); /* C_v, Eq.9  */
    st[5] = Hn[1] * (1.0 - sbar[1]); /* C_a, Eq.10 */
    st[6] = (Kall > 1 && S > 0.0) ? H / log((double)Kall) : 0.0;
    st[7] = Kall > 0 ? s_sum_all / ((double)Kall * p->Hkv) : 0.0;
    free(A_all);
  }
  return 0;
}

/* ---- O6b: per-layer totals (Eq.13-14; R19, R20) ------------------------------------------
 * C^(l) = Hn_all (1 - sbar_all); pi = softmax_l(C/T); b_l = pi_l * total.
 * Clamp to [B_min,B_max] (if budget_max > 0): layers beyond the bound on the side with the larger total violation
 * are fixed at that bound and the remaining total is re-split over the free layers in proportion to pi, until
 * nothing moves (so that sum_l B^(l) = total whenever L*B_min <= total <= L*B_max).
 * Integerise by largest remainder, ties -> lowest layer, never above B_max.  If the clamps make the
 * total unreachable every layer sits at the nearer bound. */
int omnimem_ref_layer_budgets(const omnimem_ref_params* p, const double* stats, int64_t total,
                              int32_t* layer_budget) {
  const int L = p->L;
  double* pi = (double*)malloc(sizeof(double) * L);
  double* b = (double*)malloc(sizeof(double) * L);
  int* fixed = (int*)calloc(L, sizeof(int));
  const int clamp = p->budget_max > 0;
  const double lo = clamp ? (double)p->budget_min : 0.0, hi = clamp ? (double)p->budget_max : INFINITY;
  double mx = -INFINITY, Zs = 0.0;
  for (int l = 0; l < L; ++l) {
    pi[l] = stats[l * 8 + 6] * (1.0 - stats[l * 8 + 7]) / p->temperature;
    if (pi[l] > mx) mx = pi[l];
  }
  for (int l = 0; l < L; ++l) Zs += (pi[l] = exp(pi[l] - mx));
  for (int l = 0; l < L; ++l) pi[l] /= Zs;
  if (clamp && (double)total >= hi * L) {
    for (int l = 0; l < L; ++l) layer_budget[l] = (int32_t)p->budget_max;
  } else if (clamp && (double)total <= lo * L) {
    for (int l = 0; l < L; ++l) layer_budget[l] = (int32_t)p->budget_min;
  } else {
    for (int it = 0; it <= L; ++it) {
      double rem = (double)total, pfree = 0.0;
      for (int l = 0; l < L; ++l) {
        if (fixed[l]) rem -= b[l];
        else pfree += pi[l];
      }
      int moved = 0;
      double below = 0.0, above = 0.0;
      for (int l = 0; l < L; ++l)
        if (!fixed[l]) {
          b[l] = pfree > 0.0 ? rem * pi[l] / pfree : 0.0;
          if (b[l] < lo) below += lo - b[l];
          if (b[l] > hi) above += b[l] - hi;
        }
      /* fix only the side that violates more: fixing both at once could strand budget (sum invariant, R20) */
      for (int l = 0; l < L; ++l)
        if (!fixed[l] && ((above >= below && b[l] > hi) || (above < below && b[l] < lo))) {
          b[l] = above >= below ? hi : lo;
          fixed[l] = 1;
          moved = 1;
        }
      if (!moved) break;
    }
    int64_t sum = 0;
    for (int l = 0; l < L; ++l) {
      layer_budget[l] = (int32_t)floor(b[l]);
      sum += layer_budget[l];
    }
    for (int64_t left = total - sum; left > 0; --left) {
      int best = -1;
      double bf = -1.0;
      for (int l = 0; l < L; ++l) {
        const double frac = b[l] - floor(b[l]);
        if ((double)layer_budget[l] <= floor(b[l]) && (double)layer_budget[l] + 1.0 <= hi && frac > bf) {
          bf = frac;
          best = l;
        }
      }
      if (best < 0) break;
      layer_budget[best] += 1;
    }
  }
  free(pi);
  free(b);
  free(fixed);
  return 0;
}

/* ---- O6a: modality split (Eq.11-12) -------------------------------------
 * w_v = r C_v / (r C_v + C_a); both C zero => the prior r/(r+1).  Nothing to evict (K_v+K_a <= B) => keep all.
 * Else M_v = round-half-up(w_v B) clamped so that neither modality is given more rows than it has
 * (the surplus spills to the other one), M_a = B - M_v (R22). */
int omnimem_ref_allocate(const omnimem_ref_params* p, const double* stats, const int32_t* n_v, const int32_t* n,
                         const int32_t* layer_budget, int32_t* M_v, int32_t* M_a) {
  for (int l = 0; l < p->L; ++l) {
    const int Kv = seg_len(p, n_v[l], n[l], 0), Ka = seg_len(p, n_v[l], n[l], 1);
    const int B = layer_budget[l];
    const double Cv = stats[l * 8 + 4], Ca = stats[l * 8 + 5];
    const double den = p->ratio_r * Cv + Ca;
    const double wv = den > 0.0 ? p->ratio_r * Cv / den : p->ratio_r / (p->ratio_r + 1.0);
    if (B < 0) return -1;
    if (Kv + Ka <= B) {
      M_v[l] = Kv;
      M_a[l] = Ka;
      continue;
    }
    int64_t mv = (int64_t)floor(wv * (double)B + 0.5);
    const int64_t lo = B - Ka > 0 ? B - Ka : 0, hi = Kv < B ? Kv : B;
    if (mv < lo) mv = lo;
    if (mv > hi) mv = hi;
    M_v[l] = (int32_t)mv;
    M_a[l] = (int32_t)(B - mv);
  }
  return 0;
}

/* ---- O7: Select (Eq.4-5; "top K pairs that have the highest score") -----------
 * Per (l,h,m): order the segment's indices by psi (the fp32 array) descending, equal psi by index ascending
 * (= a stable descending sort: lowest index wins ties, R23); keep the first M_m; emit them ascending. */
static int cmp_desc_stable(const void* x, const void* y, void* key) {
  const float* sort_key = (const float*)key;
  const int32_t i = *(const int32_t*)x, j = *(const int32_t*)y;
  if (sort_key[i] > sort_key[j]) return -1;
  if (sort_key[i] < sort_key[j]) return 1;
  return (i > j) - (i < j);
}
static int cmp_int_asc(const void* x, const void* y) {
  const int32_t i = *(const int32_t*)x, j = *(const int32_t*)y;
  return (i > j) - (i < j);
}

int omnimem_ref_select(const omnimem_ref_params* p, const float* psi_v, const float* psi_a, const int32_t* n_v,
                       const int32_t* n, const int32_t* M_v, const int32_t* M_a, int32_t* idx_v, int32_t* idx_a,
                       int32_t idx_cap) {
  for (int l = 0; l < p->L; ++l)
    for (int h = 0; h < p->Hkv; ++h)
      for (int m = 0; m < 2; ++m) {
        const int Km = seg_len(p, n_v[l], n[l], m);
        const int M = m == 0 ? M_v[l] : M_a[l];
        const int cap = m == 0 ? p->seg_cap_v : p->seg_cap_a;
        int32_t* out = (m == 0 ? idx_v : idx_a) + IDX3(l, h, 0, p->Hkv, idx_cap);
        if (M < 0 || M > Km || M > idx_cap) return -1;
        int32_t* order = (int32_t*)malloc(sizeof(int32_t) * (size_t)(Km + 1));
        for (int t = 0; t < Km; ++t) order[t] = t;
        const float* sort_key = (m == 0 ? psi_v : psi_a) + IDX3(l, h, 0, p->Hkv, cap);
        qsort_r(order, (size_t)Km, sizeof(int32_t), cmp_desc_stable, (void*)sort_key);
        qsort(order, (size_t)M, sizeof(int32_t), cmp_int_asc);
        for (int t = 0; t < M; ++t) out[t] = order[t];
        for (int t = M; t < idx_cap; ++t) out[t] = -1;
        free(order);
      }
  return 0;
}

/* ---- O8: prune / compaction ("pruned to a fixed size") -------------------------
 * dst[l,h,0:M_v] = visual rows idx_v, dst[l,h,M_v:M_v+M_a] = audio rows idx_a, for K and V, byte for byte;
 * n_v <- M_v, n <- M_v + M_a.  Buffers are raw bytes (row_bytes = D * element size). */
int omnimem_ref_compact(const omnimem_ref_params* p, int64_t row_bytes, const uint8_t* src_cacheX,
                        const uint8_t* chunkX, const int32_t* n_v, const int32_t* n, const int32_t* idx_v,
                        const int32_t* idx_a, int32_t idx_cap, const int32_t* M_v, const int32_t* M_a,
                        uint8_t* dst_cacheX, int32_t* n_v_out, int32_t* n_out) {
  const int Nn = p->Nn_v + p->Nn_a;
  for (int l = 0; l < p->L; ++l) {
    if (M_v[l] + M_a[l] > p->cache_cap) return -5;
    for (int h = 0; h < p->Hkv; ++h)
      for (int m = 0; m < 2; ++m) {
        const int M = m == 0 ? M_v[l] : M_a[l];
        const int32_t* idx = (m == 0 ? idx_v : idx_a) + IDX3(l, h, 0, p->Hkv, idx_cap);
        for (int jj = 0; jj < M; ++jj) {
          const int k = seg_to_logical(p, n_v[l], n[l], m, idx[jj]);
          const uint8_t* src = k < n[l] ? src_cacheX + IDX3(l * p->Hkv + h, k, 0, p->cache_cap, row_bytes)
                                        : chunkX + IDX3(l * p->Hkv + h, k - n[l], 0, Nn, row_bytes);
          uint8_t* dst = dst_cacheX + IDX3(l * p->Hkv + h, (m == 0 ? 0 : M_v[l]) + jj, 0, p->cache_cap, row_bytes);
          memcpy(dst, src, (size_t)row_bytes);
        }
      }
    n_v_out[l] = M_v[l];
    n_out[l] = M_v[l] + M_a[l];
  }
  return 0;
}

int omnimem_ref_num_threads(void) {
  int nt = 1;
#ifdef _OPENMP
#pragma omp parallel
  {
#pragma omp single
    nt = omp_get_num_threads();
  }
#endif
  return nt;
}
