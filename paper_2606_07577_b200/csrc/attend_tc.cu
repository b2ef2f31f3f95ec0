// The chunk's attention forward (Eq.1, Eq.2) for bf16, head_dim 128, on tcgen05 / TMEM / TMA (sm_100a):
//     Y_c = MHSA(Q_c, [K_v ; K_a ; K_c], [V_v ; V_a ; V_c]),   and the row log-sum-exp of its softmax.
// It is the step BEFORE the compression path: the LSE it writes is what Eq.6's column sums
// need, so a caller that runs this forward passes `lse` to omnimem_compress_chunk and score pass 1 disappears.
//
// PERSISTENT CTAs (one per SM; cfg.score_ctas overrides) draw work items from a device counter through a two-slot
// shared-memory queue, as in score_tc.cu; the K / V ring, the S / P / O barriers of each sub-tile and all their phases run on
// across items; the next item's Q tiles are loaded as soon as the current item's last S product has been issued, and its
// first S products run under the current item's epilogue.
// One item = 256 queries of one query head = two 128-row sub-tiles that take turns on the tensor pipe:
//   S_s = Q_s K_j^T   (SS mode: Q from shared memory, staged once; K tiles stream through a 4-slot ring shared with V)
//   softmax threads (one per query row): P = 2^(c2 S - m) in fp32, row sum l in fp32, P rounded to bf16 and written
//   back into tensor memory ON TOP of S_s (columns [0, 64) of its 128)
//   O_s += P_s V_j    (TS mode: P from tensor memory, V tile MN-major from shared memory)
// Issue order on the tensor pipe: O_0(j), S_0(j+1), O_1(j), S_1(j+1): while one sub-tile's softmax runs, the other's
// two products execute.  Tensor memory: S_0, S_1 at columns [0, 256), O_0, O_1 at [256, 512).
// The running reference m is LAZY, as in score pass 1: a tile's exponentials are taken against m as it stands; only if
// that could overflow (tile sum not below 2^100) the thread takes the exact path: tile maximum, new reference, and a
// rescale of its O row in tensor memory (possible because nothing of this sub-tile is in flight at that point).
// Warp roles: 0 = TMA producer + item scheduler, 1 = MMA issuer, 2 = TMEM allocator, 4-11 = softmax / epilogue (sub-tile x
// lane quarter).
#include <cuda.h>
#include <math.h>

#include <type_traits>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace omnimem {

namespace {

constexpr int kT = 128;               // rows per tile (queries per sub-tile, keys per streamed tile) and head_dim
constexpr int kTileB = kT * 128 * 2;  // 32 KB: two 64-element K-blocks of 16 KB
constexpr int kSlots = 4;             // ring of K / V tiles: K_j, V_j, K_{j+1}, V_{j+1}
constexpr int kThr = 384;             // 4 control warps + 8 softmax warps
constexpr int kOffQ = 0;                          // [2 sub][32 KB]
constexpr int kOffKV = 2 * kTileB;                // [kSlots][32 KB]
constexpr int kOffBar = kOffKV + kSlots * kTileB;
constexpr size_t kSmem = 1024 + kOffBar + 256;   // barriers, item queue and the tensor-memory slot: 180 bytes
constexpr uint32_t kColS = 0, kColO = 256;        // tensor-memory columns
constexpr int kPolyNum = 2, kPolyDen = 8;   // exponential pairs on the FMA-pipe polynomial, of every 8

// D = f32, A = B = bf16, N = 128, M = 128; bit 16: B is MN-major (the V tile: rows = keys, head_dim contiguous)
constexpr uint32_t kIdescQK = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kT >> 3) << 17) | ((uint32_t)(kT >> 4) << 24);
constexpr uint32_t kIdescPV = kIdescQK | (1u << 16);

struct AttendArgs {
  StepParams p;
  __nv_bfloat16* y;   // [L, Hq, Nn, 128]
  float* lse_nat;     // [L, Hq, Nn]
  int nx, ny, n_items;   // item grid (x = 256-query block, y = query head, z = layer), x fastest
  int* counter;          // zeroed by the launcher
};

// What one item is, computed identically by every role.
struct AItem {
  int l, jh, h, row0, n, nct, nnt, ntiles;
  int nt[2];
};
__device__ __forceinline__ void make_item(const AttendArgs& a, int item, AItem& w) {
  const StepParams& p = a.p;
  const int bx = a.nx - 1 - item % a.nx;          // the longest items (most visible chunk tiles) of a head first
  const int yz = item / a.nx;
  w.jh = yz % a.ny;
  w.l = yz / a.ny;
  w.h = w.jh / p.G;
  w.n = uniform(p.n[w.l]);
  w.row0 = bx * 2 * kT;                           // first query of this item
  w.nct = (w.n + kT - 1) / kT;                    // cache tiles
  w.nnt = (p.Nn + kT - 1) / kT;                   // chunk tiles
  for (int s = 0; s < 2; ++s) {
    const int r0 = w.row0 + s * kT;
    w.nt[s] = r0 < p.Nn ? w.nct + (p.causal ? min(w.nnt, r0 / kT + 1) : w.nnt) : 0;   // R3: chunk key t visible iff t <= i
  }
  w.ntiles = max(w.nt[0], w.nt[1]);
}

__device__ __forceinline__ void tc_ld32x(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tc_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
               :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
                  "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {   // element 2c in the low half: the A-operand word
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}

__global__ void __launch_bounds__(kThr, 1)
attend_tc_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapKc,
                 const __grid_constant__ CUtensorMap mapKn, const __grid_constant__ CUtensorMap mapVc,
                 const __grid_constant__ CUtensorMap mapVn, const AttendArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const StepParams& p = a.p;

  const uint32_t s_raw = smem_u32(smem_raw);
  const uint32_t sBase = (s_raw + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sBase - s_raw);
  const uint32_t sQ = sBase + kOffQ, sKV = sBase + kOffKV, bars = sBase + kOffBar;
  const uint32_t bar_q = bars, bar_full = bars + 8, bar_empty = bar_full + 8 * kSlots;
  const uint32_t bar_s = bar_empty + 8 * kSlots, bar_p = bar_s + 16, bar_o = bar_p + 16;
  const uint32_t bar_qfree = bar_o + 16, bar_ofree = bar_qfree + 8;                 // Q tiles / O accumulators of the last item consumed
  const uint32_t bar_qfull = bar_ofree + 16, bar_qempty = bar_qfull + 16, sQueue = bar_qempty + 16;   // item queue [2]
  uint32_t* tmem_slot = (uint32_t*)(smem + kOffBar + 8 + 16 * kSlots + 48 + 8 + 16 + 32 + 8);
  const int warp = uniform(threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(bar_q, 1);
    mbar_init(bar_qfree, 1);
    for (int i = 0; i < kSlots; ++i) { mbar_init(bar_full + 8 * i, 1); mbar_init(bar_empty + 8 * i, 1); }
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar_s + 8 * s, 1); mbar_init(bar_p + 8 * s, 4); mbar_init(bar_o + 8 * s, 1); mbar_init(bar_ofree + 8 * s, 4);
      mbar_init(bar_qfull + 8 * s, 1); mbar_init(bar_qempty + 8 * s, 9);     // consumers: the MMA warp + 8 softmax warps
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = (uint32_t)uniform((int)*tmem_slot);

  int qi = 0, qph = 0;      // consumer side of the item queue
  auto next_item = [&]() -> int {
    mbar_wait(bar_qfull + 8 * qi, qph);
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(sQueue + 4 * qi) : "memory");
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_qempty + 8 * qi);
    if (++qi == 2) { qi = 0; qph ^= 1; }
    return uniform((int)v);
  };

  if (warp == 0) {
    // ===================== TMA producer: per item Q (once the last item's S products are through), then K_0, V_0, K_1, ... =====================
    int slot = 0, ph = 1, pq = 0, pqph = 1, qfph = 1;
    for (;;) {
      mbar_wait(bar_qempty + 8 * pq, pqph);
      int item = 0;
      if (lane == 0) {
        item = atomicAdd(a.counter, 1);
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(sQueue + 4 * pq), "r"(item) : "memory");
        mbar_arrive(bar_qfull + 8 * pq);
      }
      item = uniform(item);
      if (++pq == 2) { pq = 0; pqph ^= 1; }
      if (item >= a.n_items) break;
      AItem w;
      make_item(a, item, w);
      const int lhq = w.l * p.Hq + w.jh, lhk = w.l * p.Hkv + w.h;
      mbar_wait(bar_qfree, qfph);       // every S product of the previous item has read its Q tiles
      qfph ^= 1;
      if (elect_one()) {
        mbar_expect_tx(bar_q, (w.nt[1] > 0 ? 2 : 1) * kTileB);
        for (int s = 0; s < 2; ++s)
          if (w.nt[s] > 0)
            for (int kb = 0; kb < 2; ++kb) tma_load_3d(sQ + s * kTileB + kb * (kTileB / 2), &mapQ, kb * 64, w.row0 + s * kT, lhq, bar_q);
      }
      __syncwarp();
      for (int j = 0; j < w.ntiles; ++j) {
        const bool cache = j < w.nct;
        const int r0 = (cache ? j : j - w.nct) * kT;
        for (int t = 0; t < 2; ++t) {   // t = 0: K tile, t = 1: V tile
          mbar_wait(bar_empty + 8 * slot, ph);
          if (elect_one()) {
            mbar_expect_tx(bar_full + 8 * slot, kTileB);
            const CUtensorMap* m = t == 0 ? (cache ? &mapKc : &mapKn) : (cache ? &mapVc : &mapVn);
            for (int kb = 0; kb < 2; ++kb) tma_load_3d(sKV + slot * kTileB + kb * (kTileB / 2), m, kb * 64, r0, lhk, bar_full + 8 * slot);
          }
          __syncwarp();
          if (++slot == kSlots) { slot = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    int slot = 0, ph = 0;             // ring position of the next tile to consume (K_0, V_0, K_1, ...)
    int done[2] = {0, 0};             // tiles of sub-tile s completed in earlier items: phase of its S / P / O barriers
    int items_s[2] = {0, 0};          // items in which sub-tile s had rows: phase of its O-free barrier
    int qph_mma = 0;
    auto advance = [&]() { if (++slot == kSlots) { slot = 0; ph ^= 1; } };
    for (;;) {
      const int item = next_item();
      if (item >= a.n_items) break;
      AItem w;
      make_item(a, item, w);
      const int n = w.n, nct = w.nct, ntiles = w.ntiles;
      auto issue_s = [&](int s, int kslot) {   // S_s = Q_s K^T
        if (elect_one()) {
          const uint64_t a_desc = umma_desc_sw128(sQ + s * kTileB), b_desc = umma_desc_sw128(sKV + kslot * kTileB);
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint64_t koff = (uint64_t)(((kk >> 2) * (kTileB / 2) + (kk & 3) * 32) >> 4);
            tc_mma_bf16(tmem_base + kColS + s * kT, a_desc + koff, b_desc + koff, kIdescQK, kk > 0 ? 1u : 0u);
          }
          tc_commit(bar_s + 8 * s);
        }
        __syncwarp();
      };
      auto issue_o = [&](int s, int vslot, int j) {   // O_s += P_s V
        mbar_wait(bar_p + 8 * s, (done[s] + j) & 1);
        if (j == 0) mbar_wait(bar_ofree + 8 * s, (items_s[s] & 1) ^ 1);   // the last item's epilogue has read O_s
        tc_fence_after();
        if (elect_one()) {
          const uint64_t b_desc = umma_desc_sw128_mn(sKV + vslot * kTileB, kTileB / 2);
#pragma unroll
          for (int kk = 0; kk < 8; ++kk)   // 16 keys per step: 8 TMEM columns of P, 16 rows (2048 B) of the V tile
            tc_mma_bf16_ts(tmem_base + kColO + s * kT, tmem_base + kColS + s * kT + kk * 8, b_desc + (uint64_t)((kk * 2048) >> 4),
                           kIdescPV, (j > 0 || kk > 0) ? 1u : 0u);
          tc_commit(bar_o + 8 * s);
        }
        __syncwarp();
      };
      mbar_wait(bar_q, qph_mma);
      qph_mma ^= 1;
      mbar_wait(bar_full + 8 * slot, ph);   // K_0
      tc_fence_after();
      for (int s = 0; s < 2; ++s) if (w.nt[s] > 0) issue_s(s, slot);
      if (ntiles == 1) { if (elect_one()) tc_commit(bar_qfree); __syncwarp(); }   // (no further S product in this item)
      if (elect_one()) tc_commit(bar_empty + 8 * slot);
      __syncwarp();
      advance();
      for (int j = 0; j < ntiles; ++j) {
        const int vslot = slot, vph = ph;
        advance();
        const int kslot = slot;
        mbar_wait(bar_full + 8 * vslot, vph);   // V_j
        if (j == nct - 1 && (n & (kT - 1)) != 0) {
          // the last cache tile is ragged: rows >= n of the V tile are stale cache rows.  Their P columns are zero, but
          // 0 * (Inf or NaN bits) would poison O: zero those rows in shared memory (a row is one 128-byte line per K-block)
          const int first = n - j * kT;
          for (int idx = lane; idx < (kT - first) * 16; idx += 32) {
            const int r = first + (idx >> 4), c = idx & 15;
            const uint32_t addr = sKV + vslot * kTileB + (c >> 3) * (kTileB / 2) + r * 128 + (c & 7) * 16;
            asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(addr), "r"(0) : "memory");
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
        }
        tc_fence_after();
        // ORDERING ASSUMPTION: S_s(j+1) below overwrites the tensor-memory columns that hold P_s(j), which the O_s(j) product
        // issued just before it reads as its A operand -- two tcgen05.mma on DIFFERENT accumulators with a write-after-read
        // between them, nothing waiting in between.  It relies on the tensor pipe executing one thread's tcgen05 stream in
        // issue order (see the note at the stationary copies in score_tc.cu; the PTX ISA guarantees the order only for a
        // shared accumulator).  Guarded by the multi-item attend tests (distinct P per tile, 1-5 persistent CTAs).
        if (j < w.nt[0]) issue_o(0, vslot, j);
        if (j + 1 < ntiles) { mbar_wait(bar_full + 8 * kslot, ph); tc_fence_after(); }   // K_{j+1}
        if (j + 1 < w.nt[0]) issue_s(0, kslot);
        if (j < w.nt[1]) issue_o(1, vslot, j);
        if (elect_one()) tc_commit(bar_empty + 8 * vslot);
        __syncwarp();
        if (j + 1 < w.nt[1]) issue_s(1, kslot);
        if (j + 2 == ntiles) { if (elect_one()) tc_commit(bar_qfree); __syncwarp(); }   // the item's last S products are issued
        if (j + 1 < ntiles) {
          if (elect_one()) tc_commit(bar_empty + 8 * kslot);
          __syncwarp();
          advance();
        }
      }
      for (int s = 0; s < 2; ++s) { done[s] += w.nt[s]; items_s[s] += w.nt[s] > 0 ? 1 : 0; }
    }
  } else if (warp >= 4) {
    // ===================== softmax / epilogue: thread = one query row of sub-tile s =====================
    const int s = (warp - 4) >> 2, q4 = warp & 3;
    const int r = q4 * 32 + lane;
    const float c2 = p.scale_log2e;
    const uint32_t t_lane = tmem_base + ((uint32_t)(q4 * 32) << 16);
    const uint32_t tS = t_lane + kColS + s * kT, tO = t_lane + kColO + s * kT;
    int done = 0;                     // tiles of this sub-tile completed in earlier items: phase of its S / P / O barriers
    for (;;) {
    const int item = next_item();
    if (item >= a.n_items) break;
    AItem w;
    make_item(a, item, w);
    const int n = w.n, nct = w.nct, i = w.row0 + s * kT + r;
    const int lhq = w.l * p.Hq + w.jh;
    const int nts = uniform(s == 0 ? w.nt[0] : w.nt[1]);
    if (nts > 0) {
      float m_ref = -INFINITY, lsum = 0.f;
      for (int j = 0; j < nts; ++j) {
        int limit;                               // visible key columns of this tile for this row
        if (j < nct) limit = n - j * kT;
        else {
          const int t0 = (j - nct) * kT;
          limit = p.Nn - t0;
          if (p.causal) limit = min(limit, i - t0 + 1);
        }
        mbar_wait(bar_s + 8 * s, (done + j) & 1);
        tc_fence_after();
        uint32_t pk[64];                         // the tile's P row, bf16 pairs
        float tsum, pmax;
        // exponentials of the tile against reference `mref`; fills pk, returns the fp32 row sum.  The 128 columns come in
        // four tcgen05.ld of 32: the next one is in flight while the current one is computed (wait::ld waits for all
        // outstanding loads, hence: wait, issue the next, compute).  Scale and sums are packed fp32x2; kPolyNum of every
        // kPolyDen pairs take the FMA-pipe polynomial (tc_ptx.cuh) instead of the MUFU.
        auto exp_tile = [&](float mref, auto masked_tag) {
          constexpr bool kMasked = decltype(masked_tag)::value;
          uint64_t zA = 0ull, zB = 0ull;
          const uint64_t c2c2 = pack2(c2, c2), nm = pack2(-mref, -mref);
          pmax = -INFINITY;   // largest raw score of a polynomial lane: unlike the MUFU, the polynomial does not overflow to inf
          uint32_t va[32], vb[32];
          tc_ld32x(tS, va);
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            tc_wait_ld();
            uint32_t (&cur)[32] = (c & 1) ? vb : va;
            if (c < 3) tc_ld32x(tS + (c + 1) * 32, (c & 1) ? va : vb);
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
              if (pair_is_poly_t<kPolyNum, kPolyDen>(c * 16 + e / 2)) pmax = fmaxf(pmax, fmaxf(__uint_as_float(cur[e]), __uint_as_float(cur[e + 1])));
              if (pair_is_poly_t<kPolyNum, kPolyDen>(c * 16 + e / 2 + 1)) pmax = fmaxf(pmax, fmaxf(__uint_as_float(cur[e + 2]), __uint_as_float(cur[e + 3])));
              uint64_t P01 = ex2_pair_t<kPolyNum, kPolyDen>(fma2(pack2u(cur[e], cur[e + 1]), c2c2, nm), c * 16 + e / 2);
              uint64_t P23 = ex2_pair_t<kPolyNum, kPolyDen>(fma2(pack2u(cur[e + 2], cur[e + 3]), c2c2, nm), c * 16 + e / 2 + 1);
              float p0, p1, p2, p3;
              unpack2(P01, p0, p1);
              unpack2(P23, p2, p3);
              if (kMasked) {
                const int col = c * 32 + e;
                p0 = col < limit ? p0 : 0.f; p1 = col + 1 < limit ? p1 : 0.f;
                p2 = col + 2 < limit ? p2 : 0.f; p3 = col + 3 < limit ? p3 : 0.f;
                P01 = pack2(p0, p1);
                P23 = pack2(p2, p3);
              }
              zA = add2z(zA, P01);
              zB = add2z(zB, P23);
              pk[c * 16 + e / 2] = pack_bf16(p0, p1);
              pk[c * 16 + e / 2 + 1] = pack_bf16(p2, p3);
            }
          }
          float z0, z1, z2, z3;
          unpack2(zA, z0, z1);
          unpack2(zB, z2, z3);
          return (z0 + z1) + (z2 + z3);
        };
        auto exp_tile_any = [&](float mref) {   // the unmasked body for whole tiles (warp-uniform choice)
          return __all_sync(0xffffffffu, limit >= kT) ? exp_tile(mref, std::false_type{}) : exp_tile(mref, std::true_type{});
        };
        bool ok = false;
        if (j > 0) {                             // lazy reference: exact unless something overflows
          tsum = exp_tile_any(m_ref);
          ok = tsum < 1.2676506e30f && lsum < 1.2676506e30f &&   // 2^100; false for inf and NaN
               fmaf(pmax, c2, -m_ref) < 100.f;
        }
        if (!__all_sync(0xffffffffu, ok)) {      // first tile, or the row's maximum jumped: exact path (warp-uniform)
          float mx = -INFINITY;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t v[32];
            tc_ld32x(tS + c * 32, v);
            tc_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) mx = fmaxf(mx, c * 32 + e < limit ? __uint_as_float(v[e]) : -INFINITY);
          }
          const float m_new = fmaxf(m_ref, mx * c2);
          if (j > 0) {
            // everything issued for this sub-tile has completed (S_s(j) is there, the tensor pipe runs in order) and
            // O_s(j) waits for this thread: the O row can be rescaled in place
            const float sc = ex2(m_ref - m_new);
            lsum *= sc;
            mbar_wait(bar_o + 8 * s, (done + j - 1) & 1);
            tc_fence_after();
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              uint32_t v[32];
              tc_ld32x(tO + c * 32, v);
              tc_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) v[e] = __float_as_uint(__uint_as_float(v[e]) * sc);
              tc_st32(tO + c * 32, v);
            }
          }
          m_ref = m_new;
          tsum = exp_tile_any(m_ref);
        }
        lsum += tsum;
#pragma unroll
        for (int c = 0; c < 4; ++c) tc_st16(tS + c * 16, pk + c * 16);   // P over the first 64 columns of S
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_p + 8 * s);
      }
      // epilogue: Y = O / l (bf16), lse = ln 2 (m + log2 l)
      mbar_wait(bar_o + 8 * s, (done + nts - 1) & 1);
      tc_fence_after();
      const float inv = 1.f / lsum;
      const bool valid = i < p.Nn;
      uint4* yrow = reinterpret_cast<uint4*>(a.y + ((long long)lhq * p.Nn + (valid ? i : 0)) * kT);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t v[32];
        tc_ld32x(tO + c * 32, v);
        tc_wait_ld();
        if (c == 3) {                            // O_s is in registers: the next item's first P V product may overwrite it
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_ofree + 8 * s);
        }
        if (valid) {
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            uint4 o;
            o.x = pack_bf16(__uint_as_float(v[8 * u]) * inv, __uint_as_float(v[8 * u + 1]) * inv);
            o.y = pack_bf16(__uint_as_float(v[8 * u + 2]) * inv, __uint_as_float(v[8 * u + 3]) * inv);
            o.z = pack_bf16(__uint_as_float(v[8 * u + 4]) * inv, __uint_as_float(v[8 * u + 5]) * inv);
            o.w = pack_bf16(__uint_as_float(v[8 * u + 6]) * inv, __uint_as_float(v[8 * u + 7]) * inv);
            yrow[c * 4 + u] = o;
          }
        }
      }
      if (valid) a.lse_nat[(long long)lhq * p.Nn + i] = (m_ref + log2f(lsum)) * 0.6931471805599453f;
      done += nts;
    }
    }  // work items
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// [outer, rows, 128] bf16 row-major -> 3-D map, box = 64 x 128 x 1, 128-byte swizzle, zero fill out of bounds
cudaError_t make_map(EncodeTiledFn enc, CUtensorMap* m, const void* base, uint64_t rows, uint64_t outer) {
  if (rows == 0 || outer == 0 || base == nullptr) { memset(m, 0, sizeof(*m)); return cudaSuccess; }
  const cuuint64_t dims[3] = {128, rows, outer};
  const cuuint64_t strides[2] = {256, rows * 256};
  const cuuint32_t box[3] = {64, (cuuint32_t)kT, 1};
  const cuuint32_t es[3] = {1, 1, 1};
  const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_attend_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, void* y, float* lse_nat,
                             cudaStream_t st, int* launches) {
  if (p.Nn == 0) return cudaSuccess;
  omnimem_ctx* c = const_cast<omnimem_ctx*>(ctx);
  if (!c->encode_tiled) {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q);
    if (e != cudaSuccess) return e;
    if (q != cudaDriverEntryPointSuccess || !f) return cudaErrorNotSupported;
    c->encode_tiled = f;
  }
  EncodeTiledFn enc = (EncodeTiledFn)c->encode_tiled;
  CUtensorMap mq, mkc, mkn, mvc, mvn;
  cudaError_t e;
  if ((e = make_map(enc, &mq, b.Q, p.Nn, (uint64_t)p.L * p.Hq)) != cudaSuccess) return e;
  if ((e = make_map(enc, &mkc, b.cacheK, p.cache_cap, (uint64_t)p.L * p.Hkv)) != cudaSuccess) return e;
  if ((e = make_map(enc, &mkn, b.chunkK, p.Nn, (uint64_t)p.L * p.Hkv)) != cudaSuccess) return e;
  if ((e = make_map(enc, &mvc, b.cacheV, p.cache_cap, (uint64_t)p.L * p.Hkv)) != cudaSuccess) return e;
  if ((e = make_map(enc, &mvn, b.chunkV, p.Nn, (uint64_t)p.L * p.Hkv)) != cudaSuccess) return e;
  AttendArgs a{};
  a.p = p;
  a.y = (__nv_bfloat16*)y;
  a.lse_nat = lse_nat;
  a.nx = (p.Nn + 2 * kT - 1) / (2 * kT);
  a.ny = p.Hq;
  a.n_items = a.nx * p.Hq * p.L;
  a.counter = ctx->sched + 2;
  e = cudaFuncSetAttribute(attend_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem);
  if (e != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(a.counter, 0, sizeof(int), st)) != cudaSuccess) return e;
  const int ctas = ctx->cfg.score_ctas > 0 && ctx->cfg.score_ctas < ctx->sm_count ? ctx->cfg.score_ctas : ctx->sm_count;
  ++*launches;
  attend_tc_kernel<<<a.n_items < ctas ? a.n_items : ctas, kThr, kSmem, st>>>(mq, mkc, mkn, mvc, mvn, a);
  return cudaGetLastError();
}

}  // namespace omnimem
