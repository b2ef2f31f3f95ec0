// tcgen05 / TMEM / TMA scoring kernels for bf16, head_dim 128 (sm_100a only).
//
// Eq.6 needs the softmax row normaliser before the column sums, so the QK^T contraction runs twice:
//   pass 1 (kPass == 1)  S  = Q K^T, M = 128 queries per sub-tile: each thread owns one query row of the TMEM
//                        accumulator, keeps an online max / sum and writes lse2 = log2 sum_k 2^(c2 s_k).
//   pass 2 (kPass == 2)  S^T = K Q^T, M = 128 keys per sub-tile: each thread owns one KEY row, the sum over
//                        queries is thread-local: a_k = sum_{g,i} 2^(c2 s - lse2_i).  No atomics, no shuffles.
//   rescue (kPass == 3) pass 2's tiles once more, in the LOG domain, for the items (256 keys of one head and layer) that hold
//                        a key whose fp32 sum came out below 2^-100 (R31): each thread keeps a running maximum
//                        with its sum, la_k = log2 sum_{g,i} 2^(c2 s - lse2_i).  The items come from a device-built list, so
//                        the cost is bounded by one more pass 2 however many keys are flagged, and is ~0 when none is.
// Both kernels are PERSISTENT: one CTA per SM (cfg.score_ctas overrides the count) draws work items (256 stationary rows
// of one head and layer x their whole streamed sequence) from a device counter; the TMA stage ring, the accumulator ring,
// the lse ring and all their barrier phases run on across items, and the producer warp prefetches the next item's tiles
// while the epilogue finishes the current one.
// An item = two stationary 128-row sub-tiles.  They arrive through the same TMA ring as the streamed tiles and are copied
// into tensor memory by the MMA warp (tcgen05.cp 128x256b, 64 TMEM columns each: the A operand of a TS-mode tcgen05.mma,
// in issue order between the previous item's last MMAs and this item's first).  The other operand streams as 128-row
// tiles (B, six 32 KB stages); one elected thread issues tcgen05.mma (M=128,N=128,K=16 x 8 per tile and sub-tile) into a
// ring of three 128-column TMEM accumulators shared by both sub-tiles; four 4-warp epilogue groups (sub-tile x column
// half) drain them with tcgen05.ld 32x32b: a thread owns one row and 64 of the tile's 128 columns, frees the TMEM buffer
// as soon as its registers hold the data, and merges with its partner thread once per item.
// The epilogue is bound by the MUFU ex2 pipe, by instruction dispatch and -- over a whole step -- by the board's power
// cap: 2 of every 8 exponential pairs run as a packed fp32x2 degree-3 polynomial on the FMA pipe,
// and the tile loops carry as little else as possible.
// Warp roles: 0 = TMA producer + item scheduler, 1 = MMA issuer, 2 = TMEM allocator, 4-19 = epilogue.
#include <cuda.h>
#include <math.h>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace omnimem {

constexpr int kTile = 128;         // rows per operand tile (UMMA M and N)
constexpr int kHeadDim = 128;      // D
constexpr int kKBlock = 64;        // bf16 elements per 128-byte swizzle atom row
constexpr int kTileBytes = kTile * kHeadDim * 2;  // 32 KB: two 16 KB K-blocks

constexpr int kStages = 6;          // B ring (32 KB stages)
constexpr int kThreads = 640;       // 4 control warps + 16 epilogue warps (4 groups: sub-tile x column half)
constexpr int kTmemCols = 512;
constexpr int kAccBufs = 3;         // TMEM accumulator ring shared by both sub-tiles: columns [0, 384)
constexpr int kTmemA = kAccBufs * kTile;  // stationary operand: 64 columns per sub-tile at [384, 512)
constexpr int kLseSlots = 16;       // pass 2: ring of 128-float lse2 tiles (512 B each); see the reuse argument at the producer
constexpr int kHalf = kTile / 2;    // columns of a tile owned by one epilogue thread
constexpr int kOffLse = kStages * kTileBytes;
constexpr int kOffMerge = kOffLse + kLseSlots * kTile * 4;       // [2 item parities][2 sub][128 rows] float4
constexpr int kOffBars = kOffMerge + 2 * 2 * kTile * 16;
constexpr int kQueue = 2;           // work items announced ahead by the producer warp
constexpr size_t kSmemBytes = 1024 /*align slack*/ + kOffBars + 512 /*barriers + tmem slot*/;

constexpr int kKBlockBytes = kTile * 128;   // one 64-element K-block of a streamed tile (16 KB)
constexpr bool kLazyMax = true;   // pass 1: running reference instead of a per-tile maximum (see the loop)

// share of the exponential PAIRS of a row that run as the fp32x2 polynomial on the FMA pipe instead of on the MUFU
// (tc_ptx.cuh; measured optimum of both scoring passes under the 1000 W cap: 2 of 8, degree 3)
constexpr int kPolyNum = 2, kPolyDen = 8;
__device__ __forceinline__ constexpr bool pair_is_poly(int pi) { return pair_is_poly_t<kPolyNum, kPolyDen>(pi); }
__device__ __forceinline__ uint64_t ex2_pair(uint64_t X, int pi) { return ex2_pair_t<kPolyNum, kPolyDen>(X, pi); }

// Instruction descriptor: D = f32 (bit 4), A = B = bf16 (bits 7, 10), both K-major, N >> 3 at bit 17, M >> 4 at bit 24.
constexpr uint32_t kIdesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kTile >> 3) << 17) | ((uint32_t)(kTile >> 4) << 24);

struct TcArgs {
  StepParams p;
  float* lse2;         // [L, Hq, lse_stride] NEGATED log2-domain LSE (internal; padded rows hold -inf)
  int lse_stride;
  float* lse_nat;      // pass 1: optional natural-log output [L, Hq, Nn]
  float* row_entropy;  // pass 1: optional [L, Hq, Nn]
  float* a_v;          // pass 2 outputs
  float* a_a;
  int n_cache_pairs;   // pass 2: ceil(cache_cap / 256)
  // persistent CTAs: work item = (x, y, z) of the nx * ny * nz item grid, x fastest; handed out through *counter
  int nx, ny, n_items;
  int* counter;        // zeroed by the launcher
  // rescue (kPass == 3): the items to work on are item_list[0 .. *item_count) (device data, written by rescue_items_kernel)
  const int* item_list;
  const int* item_count;
  float* la_v;         // rescue outputs: log2 of the importance, [L, Hkv, seg_cap_m]
  float* la_a;
};

constexpr float kTinyImportance = 7.888609052210118e-31f;   // 2^-100: below it the fp32 column sum is not trusted (R31)

// What one CTA works on, computed identically by every role.
struct Work {
  int l, lhA;            // layer; outer TMA coordinate of the stationary operand
  int rowA0;             // first row of sub-tile 0 in the stationary operand
  bool a_chunk;          // pass 2: stationary keys come from the chunk (else cache)
  bool sub_valid[2];
  int ntiles;            // streamed tiles in this CTA's sequence
  // pass 1
  int n_cache_tiles, ntiles_sub[2], h;
  // pass 2
  int it0[2], tiles_per_g, hq0;
  int seq0;              // first query tile of the streamed sequence (== it0[0])
  // which accumulator batches exist for sub-tile s (copies of ntiles_sub / it0 / sub_valid made after the kernel's early
  // exit: see the note there)
  int ntp[2], it0p[2];
  bool validp[2];
  int nbatch;            // accumulator batches of the item (both sub-tiles)
};

template <int kPass>
__device__ __forceinline__ bool make_work(const TcArgs& a, Work& w, int item) {   // item: index in the (x, y, z) item grid
  const StepParams& p = a.p;
  if (kPass == 3) item = uniform(a.item_list[item]);   // position in the list of flagged items -> pass 2's item index
  int bx = item % a.nx;
  const int yz = item / a.nx, by = yz % a.ny;
  w.l = yz / a.ny;
  w.nbatch = 0;
  // values loaded from memory are made provably warp-uniform (shfl) so that the control warps stay on the uniform datapath
  const int n = uniform(p.n[w.l]);
  if (p.skip_budget != nullptr && n + p.Nn <= uniform(p.skip_budget[w.l])) return false;
  bool mine;
  if (kPass == 1) {
    bx = a.nx - 1 - bx;        // the longest items (most visible chunk tiles) of a head first
    const int j = by;          // query head
    w.h = j / p.G;
    w.lhA = w.l * p.Hq + j;
    w.rowA0 = bx * 2 * kTile;
    w.a_chunk = false;
    w.n_cache_tiles = (n + kTile - 1) / kTile;
    const int nct = (p.Nn + kTile - 1) / kTile;
    w.ntiles = 0;
    for (int s = 0; s < 2; ++s) {
      const int r0 = w.rowA0 + s * kTile;
      w.sub_valid[s] = r0 < p.Nn;
      const int nc = p.causal ? min(nct, r0 / kTile + 1) : nct;  // R3: chunk key t visible iff t <= i
      w.ntiles_sub[s] = w.sub_valid[s] ? w.n_cache_tiles + nc : 0;
      w.ntiles = max(w.ntiles, w.ntiles_sub[s]);
      w.it0[s] = 0;
    }
    w.nbatch = w.ntiles_sub[0] + w.ntiles_sub[1];
    mine = w.sub_valid[0];
  } else {
    const int h = by;  // KV head
    w.h = h;
    w.lhA = w.l * p.Hkv + h;
    w.hq0 = w.l * p.Hq + h * p.G;
    int valid_rows;
    if (bx < a.n_cache_pairs) {
      w.a_chunk = false;
      w.rowA0 = bx * 2 * kTile;
      valid_rows = n;
    } else {
      w.a_chunk = true;
      w.rowA0 = (bx - a.n_cache_pairs) * 2 * kTile;
      valid_rows = p.Nn;
    }
    const int nqt = (p.Nn + kTile - 1) / kTile;
    for (int s = 0; s < 2; ++s) {
      const int r0 = w.rowA0 + s * kTile;
      w.sub_valid[s] = r0 < valid_rows;
      w.it0[s] = (p.causal && w.a_chunk) ? r0 / kTile : 0;  // first query tile that can see this key sub-tile
      w.ntiles_sub[s] = 0;
    }
    w.seq0 = w.it0[0];
    w.tiles_per_g = nqt - w.seq0;
    w.ntiles = w.sub_valid[0] ? p.G * w.tiles_per_g : 0;
    if (w.ntiles <= 0) { w.ntiles = 0; w.sub_valid[0] = w.sub_valid[1] = false; }
    for (int s = 0; s < 2; ++s)
      if (w.sub_valid[s]) w.nbatch += p.G * (nqt - max(w.it0[s], w.seq0));
    mine = w.sub_valid[0];
  }
  for (int s = 0; s < 2; ++s) { w.ntp[s] = w.ntiles_sub[s]; w.it0p[s] = w.it0[s]; w.validp[s] = w.sub_valid[s]; }
  return mine;
}

// Steady state of pass 2 (cached keys, or no causal mask): both sub-tiles take every streamed tile and nothing is masked;
// the accumulator ring advances by two batches per tile.  The ring position comes in through shuffles so that ptxas keeps
// the loop's ring and barrier bookkeeping on the uniform datapath (254 instructions per tile and thread in the
// one-item-per-CTA kernel of round 1, 292 when the persistent kernel carried the positions in vector registers).
struct SteadyState { int buf, ph; uint64_t acc01, acc23; };
__device__ __forceinline__ SteadyState colsum_steady(int ntiles, int s, int half, int jt, uint32_t t_col, float c2, int buf, int ph,
                                                  uint64_t acc01, uint64_t acc23) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t sB = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sLse = sB + kOffLse, bars = sB + kOffBars;
  const uint32_t bar_sfull = bars + 16 * kStages, bar_sempty = bar_sfull + 8 * kAccBufs, bar_lse = bar_sempty + 8 * kAccBufs;
  const int lane = threadIdx.x & 31;
  ntiles = uniform(ntiles); s = uniform(s); half = uniform(half); jt = uniform(jt); buf = uniform(buf); ph = uniform(ph);
  const uint64_t c2c2 = pack2(c2, c2);
  // position in the lse ring, kept as loop-carried addresses (one uniform register each for the tile's 512 bytes and for
  // its barrier; computed from the tile index, ptxas split the address in two and copied one part into a vector register
  // for each of the 16 loads)
  const int slot0 = jt & (kLseSlots - 1);
  uint32_t l_addr = sLse + (uint32_t)(slot0 * kTile + half * kHalf) * 4, l_bar = bar_lse + 8 * slot0;
  const uint32_t l_bar_end = bar_lse + 8 * kLseSlots;
  int l_par = (jt / kLseSlots) & 1;
  for (int j = 0; j < ntiles; ++j) {
    int own = buf + s, oph = ph;
    if (own >= kAccBufs) { own -= kAccBufs; oph ^= 1; }
    uint32_t v0[32], v1[32];
    mbar_wait(bar_sfull + 8 * own, oph);
    tc_fence_after();
    const uint32_t t_addr = t_col + (uint32_t)(own * kTile);
    tc_ld32(t_addr, v0);
    tc_ld32(t_addr + 32, v1);
    tc_wait_ld();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_sempty + 8 * own);
    buf += 2;
    if (buf >= kAccBufs) { buf -= kAccBufs; ph ^= 1; }
    mbar_wait(l_bar, l_par);
    const uint32_t l_cur = l_addr;
    l_addr += kTile * 4;
    l_bar += 8;
    if (l_bar == l_bar_end) { l_bar = bar_lse; l_addr -= kLseSlots * kTile * 4; l_par ^= 1; }
#pragma unroll
    for (int e4 = 0; e4 < 8; ++e4) {
      const float4 la = lds128(l_cur + e4 * 16), lb = lds128(l_cur + 128 + e4 * 16);
      const uint64_t x0 = fma2(pack2u(v0[4 * e4], v0[4 * e4 + 1]), c2c2, pack2(la.x, la.y));
      const uint64_t x1 = fma2(pack2u(v0[4 * e4 + 2], v0[4 * e4 + 3]), c2c2, pack2(la.z, la.w));
      const uint64_t x2 = fma2(pack2u(v1[4 * e4], v1[4 * e4 + 1]), c2c2, pack2(lb.x, lb.y));
      const uint64_t x3 = fma2(pack2u(v1[4 * e4 + 2], v1[4 * e4 + 3]), c2c2, pack2(lb.z, lb.w));
      acc01 = add2z(acc01, ex2_pair(x0, 4 * e4));
      acc23 = add2z(acc23, ex2_pair(x1, 4 * e4 + 1));
      acc01 = add2z(acc01, ex2_pair(x2, 4 * e4 + 2));
      acc23 = add2z(acc23, ex2_pair(x3, 4 * e4 + 3));
    }
  }
  return SteadyState{buf, ph, acc01, acc23};
}

template <int kPass, bool kEntropy>
__global__ void __launch_bounds__(kThreads, 1)
score_tc_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapKc,
                const __grid_constant__ CUtensorMap mapKn, const TcArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const StepParams& p = a.p;
  const int n_items = kPass == 3 ? uniform(*a.item_count) : a.n_items;

  // 1024-byte alignment (128B swizzle) computed on the 32-bit shared-window address: the window offset of the dynamic
  // array is a link-time constant, so every barrier / stage address below folds into an immediate
  const uint32_t s_raw = smem_u32(smem_raw);
  const uint32_t sB = (s_raw + 1023u) & ~1023u;          // [kStages][2 kb][16 KB]
  uint8_t* smem = smem_raw + (sB - s_raw);
  const uint32_t sLse = sB + kOffLse;                    // [kLseSlots][128] float (pass 2)
  float4* sMerge = reinterpret_cast<float4*>(smem + kOffMerge);  // [2 item parities][2 sub][128]
  const uint32_t bars = sB + kOffBars;
  const uint32_t bar_full = bars, bar_empty = bar_full + 8 * kStages;
  const uint32_t bar_sfull = bar_empty + 8 * kStages, bar_sempty = bar_sfull + 8 * kAccBufs;  // [accumulator buffer]
  const uint32_t bar_lse = bar_sempty + 8 * kAccBufs;                           // [kLseSlots]
  const uint32_t bar_qfull = bar_lse + 8 * kLseSlots, bar_qempty = bar_qfull + 8 * kQueue;   // [kQueue] item queue
  const uint32_t sQueue = bar_qempty + 8 * kQueue;                              // [kQueue] int
  uint32_t* tmem_slot = (uint32_t*)(smem + kOffBars + 16 * kStages + 16 * kAccBufs + 8 * kLseSlots + 16 * kQueue + 4 * kQueue);

  const int warp = uniform(threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 1); }
    // an accumulator buffer is free when the 8 warps of its sub-tile's group have read it
    for (int i = 0; i < kAccBufs; ++i) { mbar_init(bar_sfull + 8 * i, 1); mbar_init(bar_sempty + 8 * i, 8); }
    for (int i = 0; i < kLseSlots; ++i) mbar_init(bar_lse + 8 * i, 1);
    // a queue slot is free again when the MMA warp and the 16 epilogue warps have read it
    for (int i = 0; i < kQueue; ++i) { mbar_init(bar_qfull + 8 * i, 1); mbar_init(bar_qempty + 8 * i, 17); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = (uint32_t)uniform((int)*tmem_slot);

  // PERSISTENT CTA: one per SM, all rings (shared-memory stages, accumulators, lse tiles) and their phases run on across
  // work items.  The producer warp draws item indices from a global counter and announces them through a two-slot queue;
  // it runs ahead of the consumers by up to kStages tiles, so the next item's stationary and first streamed tiles are in
  // shared memory before the epilogue has finished the current item.
  int qi = 0, qph = 0;      // consumer side of the item queue
  auto next_item = [&]() -> int {
    mbar_wait(bar_qfull + 8 * qi, qph);
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(sQueue + 4 * qi) : "memory");
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_qempty + 8 * qi);
    if (++qi == kQueue) { qi = 0; qph ^= 1; }
    return uniform((int)v);
  };

  if (warp < 4) {
  if (warp == 0) {
    // ===================== TMA producer: stationary sub-tiles, then the streamed operand =====================
    int stage = 0, sph = 1, slot = 0, pq = 0, pqph = 1;
    for (;;) {
      mbar_wait(bar_qempty + 8 * pq, pqph);
      int item = 0;
      if (lane == 0) {
        item = atomicAdd(a.counter, 1);
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(sQueue + 4 * pq), "r"(item) : "memory");
        mbar_arrive(bar_qfull + 8 * pq);
      }
      item = uniform(item);
      if (++pq == kQueue) { pq = 0; pqph ^= 1; }
      if (item >= n_items) break;
      Work w;
      if (!make_work<kPass>(a, w, item)) continue;
      int it = kPass != 1 ? w.seq0 : 0, g = 0;   // pass 2: query tile / group member of tile j, kept incrementally
      stage = uniform(stage); sph = uniform(sph); slot = uniform(slot);   // see the epilogue
      // the stationary sub-tiles go through the same ring: the MMA warp copies them on into tensor memory (tcgen05.cp).
      // Rows past the end of the tensor are zero-filled by the TMA unit; rows n .. cache_cap of a cache tile are stale,
      // which only reaches the (unpublished) results of those rows' own threads.
      for (int s = 0; s < 2; ++s) {
        if (!w.sub_valid[s]) continue;
        mbar_wait(bar_empty + 8 * stage, sph);
        if (elect_one()) {
          const CUtensorMap* mA = kPass == 1 ? &mapQ : (w.a_chunk ? &mapKn : &mapKc);
          mbar_expect_tx(bar_full + 8 * stage, kTileBytes);
          for (int kb = 0; kb < 2; ++kb)
            tma_load_3d(sB + stage * kTileBytes + kb * kKBlockBytes, mA, kb * kKBlock, w.rowA0 + s * kTile, w.lhA, bar_full + 8 * stage);
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; sph ^= 1; }
      }
      for (int j = 0; j < w.ntiles; ++j) {
        mbar_wait(bar_empty + 8 * stage, sph);
        const CUtensorMap* mB;
        int row0, lh;
        if (kPass == 1) {
          const bool cache = j < w.n_cache_tiles;
          mB = cache ? &mapKc : &mapKn;
          row0 = (cache ? j : j - w.n_cache_tiles) * kTile;
          lh = w.l * p.Hkv + w.h;
        } else {
          mB = &mapQ;
          row0 = it * kTile;
          lh = w.hq0 + g;
          if (++it == w.seq0 + w.tiles_per_g) { it = w.seq0; ++g; }
        }
        if (elect_one()) {
          mbar_expect_tx(bar_full + 8 * stage, kTileBytes);
          if (kPass != 1) {
            // lse2 of these 128 queries: its own ring + barrier, slot = (streamed tiles so far) % 16.  The slot was last
            // read 16 streamed tiles ago; this load is issued only after the ring entry kStages back (a streamed tile at
            // most kStages + 2 tiles back, the stationary tiles of an item boundary included) was consumed by its MMAs,
            // which needed accumulators that the epilogue releases only after it finished computing every earlier batch:
            // everything more than kStages + 2 + 3 = 11 tiles back is done.
            mbar_expect_tx(bar_lse + 8 * slot, kTile * 4);
            bulk_load(sLse + slot * kTile * 4, a.lse2 + (long long)lh * a.lse_stride + row0, kTile * 4, bar_lse + 8 * slot);
          }
          for (int kb = 0; kb < 2; ++kb)
            tma_load_3d(sB + stage * kTileBytes + kb * kKBlockBytes, mB, kb * kKBlock, row0, lh, bar_full + 8 * stage);
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; sph ^= 1; }
        if (++slot == kLseSlots) slot = 0;
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    int buf = 0, ph = 0;  // accumulator ring position of the next batch
    int stage = 0, sph = 0;
    for (;;) {
      const int item = next_item();
      if (item >= n_items) break;
      Work w;
      if (!make_work<kPass>(a, w, item)) continue;
      int it = kPass != 1 ? w.seq0 : 0;
      buf = uniform(buf); ph = uniform(ph); stage = uniform(stage); sph = uniform(sph);   // see the epilogue
      // stationary sub-tiles: shared memory -> tensor memory columns kTmemA + 64 s (lane = row, word c = elements 2c,
      // 2c+1: the A-operand layout of a TS-mode tcgen05.mma), 8 columns per K16 step.  The copies run in issue order with
      // the MMAs: after the previous item's last MMAs (which read these columns), before this item's first.
      // ORDERING ASSUMPTION (write-after-read on the A columns): nothing waits between the previous item's last TS-mode
      // MMAs and these copies.  The PTX ISA states that tcgen05.cp -> tcgen05.mma and tcgen05.mma -> tcgen05.mma issued by
      // one thread execute in issue order; for tcgen05.mma -> tcgen05.cp it makes no such statement.  This kernel relies on
      // the tensor pipe executing one thread's tcgen05.cp / .mma stream in order (what sm_100 does: block-scaled GEMM
      // mainloops in the vendor's template library refill their scale-factor columns with tcgen05.cp behind the MMAs
      // that read them in the same way).  Regression guard: test_persistent_ctas_walk_several_items and the rescue test
      // with 3 CTAs give every CTA many consecutive items with distinct stationary tiles; a reordering would corrupt the
      // second item's rows.  If a future part relaxes the order: commit the item's last MMA to a barrier of its own and
      // wait on it here before the first copy (the stage-full wait above hides most of that latency).
      for (int s = 0; s < 2; ++s) {
        if (!w.validp[s]) continue;
        mbar_wait(bar_full + 8 * stage, sph);
        tc_fence_after();
        if (elect_one()) {
          const uint64_t a_desc = umma_desc_sw128(sB + stage * kTileBytes);
#pragma unroll
          for (int kk = 0; kk < kHeadDim / 16; ++kk) {
            const uint64_t koff = (uint64_t)(((kk >> 2) * kKBlockBytes + (kk & 3) * 32) >> 4);
            tc_cp_128x256b(tmem_base + (uint32_t)(kTmemA + s * (kHeadDim / 2) + kk * 8), a_desc + koff);
          }
          tc_commit(bar_empty + 8 * stage);
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; sph ^= 1; }
      }
      for (int j = 0; j < w.ntiles; ++j) {
        mbar_wait(bar_full + 8 * stage, sph);
        tc_fence_after();
        for (int s = 0; s < 2; ++s) {
          if (!(kPass == 1 ? j < w.ntp[s] : (w.validp[s] && it >= w.it0p[s]))) continue;
          mbar_wait(bar_sempty + 8 * buf, ph ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(buf * kTile);
          const uint32_t a_tmem = tmem_base + (uint32_t)(kTmemA + s * (kHeadDim / 2));
          const uint64_t b_desc = umma_desc_sw128(sB + stage * kTileBytes);
          if (elect_one()) {
#pragma unroll
            for (int kk = 0; kk < kHeadDim / 16; ++kk) {
              // advancing the start-address field (bytes >> 4) walks K inside / across the two 64-element swizzle blocks
              const uint64_t koff = (uint64_t)(((kk >> 2) * kKBlockBytes + (kk & 3) * 32) >> 4);
              tc_mma_bf16_ts(d_tmem, a_tmem + kk * 8, b_desc + koff, kIdesc, kk > 0 ? 1u : 0u);
            }
            tc_commit(bar_sfull + 8 * buf);
          }
          __syncwarp();
          if (++buf == kAccBufs) { buf = 0; ph ^= 1; }
        }
        if (elect_one()) tc_commit(bar_empty + 8 * stage);
        __syncwarp();
        if (++stage == kStages) { stage = 0; sph ^= 1; }
        if (kPass != 1 && ++it == w.seq0 + w.tiles_per_g) it = w.seq0;
      }
    }
  }
  } else {
    // ===================== epilogue groups =====================
    const int grp = (warp - 4) >> 2;     // 0..3
    const int s = grp >> 1;              // sub-tile
    const int half = grp & 1;            // which 64 of the tile's 128 columns
    const int q4 = warp & 3;             // TMEM lane quarter this warp may touch
    const int r = q4 * 32 + lane;        // row of the sub-tile == TMEM lane
    const int col0 = half * kHalf;
    const float c2 = p.scale_log2e;
    // "this warp has read accumulator buffer b"
    auto release = [&](int b) {
      if (lane == 0) mbar_arrive(bar_sempty + 8 * b);
    };
    const uint32_t t_lane = tmem_base + ((uint32_t)(q4 * 32) << 16);
    const uint32_t t_col = t_lane + (uint32_t)col0;
    int buf = 0, ph = 0;  // accumulator ring position, advanced for every batch of either sub-tile, across work items
    int jt = 0;           // pass 2: streamed tiles of the earlier items, modulo the lse ring (slot and parity of tile j)
    int mpar = 0;         // merge buffer of this item (double-buffered: the partner reads while the next item's halves write)
    for (;;) {
    const int item = next_item();
    if (item >= n_items) break;
    Work w;
    if (!make_work<kPass>(a, w, item)) continue;
    if (!w.sub_valid[s]) {
      // This group has no rows in the item (ragged last block of a head): keep the ring positions in step, and do NOT run
      // ahead: the mbarrier waits compare phase parities, which is only sound while a waiter is less than one ring
      // revolution away from the phase it waits for.  The groups of sub-tile 0 arrive here when they are done with the item.
      for (int b = w.nbatch % (2 * kAccBufs); b > 0; --b) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } }
      jt = (jt + w.ntiles) & (2 * kLseSlots - 1);
      named_bar_sync(3, 512);
      continue;
    }
    const bool idle_partner = !w.sub_valid[1];   // (sub-tile 0 is valid in every item that is worked on)
    // loop-carried ring positions: re-derived from a shuffle at every item so that ptxas keeps them (and the barrier /
    // tensor-memory addresses computed from them) on the uniform datapath inside the tile loops
    buf = uniform(buf); ph = uniform(ph); jt = uniform(jt);
    {
      float4* sMg = sMerge + mpar * 2 * kTile;
      mpar ^= 1;
      if (kPass == 1) {
        const int i = w.rowA0 + s * kTile + r;  // query index in the chunk
        const int n = p.n[w.l];
        float m_run = -1e30f, Z = 0.f, W = 0.f;
        // accumulator batch at ring position (b, bph) -> registers; the TMEM buffer is released as soon as they hold it
        auto load_tile = [&](int b, int bph, uint32_t (&v0)[32], uint32_t (&v1)[32]) {
          mbar_wait(bar_sfull + 8 * b, bph);
          tc_fence_after();
          const uint32_t t_addr = t_col + (uint32_t)(b * kTile);
          tc_ld32(t_addr, v0);
          tc_ld32(t_addr + 32, v1);
          tc_wait_ld();
          tc_fence_before();
          __syncwarp();
          release(b);
        };
        // online softmax statistics of this thread's 64 columns of one tile; limit = visible columns (>= 64: all)
        auto row_update = [&](const uint32_t (&v0)[32], const uint32_t (&v1)[32], int limit) {
          float x[kHalf];
          if (limit >= kHalf) {
#pragma unroll
            for (int e = 0; e < 32; ++e) { x[e] = __uint_as_float(v0[e]); x[32 + e] = __uint_as_float(v1[e]); }
          } else {
#pragma unroll
            for (int e = 0; e < 32; ++e) {
              x[e] = e < limit ? __uint_as_float(v0[e]) : -INFINITY;
              x[32 + e] = 32 + e < limit ? __uint_as_float(v1[e]) : -INFINITY;
            }
          }
          float mx[4] = {x[0], x[1], x[2], x[3]};
#pragma unroll
          for (int e = 4; e < kHalf; ++e) mx[e & 3] = fmaxf(mx[e & 3], x[e]);
          const float cmax = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3]));
          const float m_new = fmaxf(m_run, cmax * c2);
          const float rs = ex2(m_run - m_new);
          m_run = m_new;
          float wz[4] = {0.f, 0.f, 0.f, 0.f};
          uint64_t z01 = 0ull, z23 = 0ull;  // packed fp32x2 partial sums
          const uint64_t c2c2 = pack2(c2, c2), nm = pack2(-m_new, -m_new);
#pragma unroll
          for (int e = 0; e < kHalf; e += 4) {
            const uint64_t A01 = fma2(pack2(x[e], x[e + 1]), c2c2, nm), A23 = fma2(pack2(x[e + 2], x[e + 3]), c2c2, nm);
            const uint64_t P01 = ex2_pair(A01, e / 2), P23 = ex2_pair(A23, e / 2 + 1);
            z01 = add2z(z01, P01);
            z23 = add2z(z23, P23);
            if (kEntropy) {  // sum p z2 over visible columns (masked ones have p = 0 but z2 = -inf)
              float a0, a1, a2, a3, p0, p1, p2, p3;
              unpack2(A01, a0, a1);
              unpack2(A23, a2, a3);
              unpack2(P01, p0, p1);
              unpack2(P23, p2, p3);
              wz[0] = fmaf(p0, limit > e ? a0 + m_new : 0.f, wz[0]);
              wz[1] = fmaf(p1, limit > e + 1 ? a1 + m_new : 0.f, wz[1]);
              wz[2] = fmaf(p2, limit > e + 2 ? a2 + m_new : 0.f, wz[2]);
              wz[3] = fmaf(p3, limit > e + 3 ? a3 + m_new : 0.f, wz[3]);
            }
          }
          float z0, z1, z2, z3;
          unpack2(z01, z0, z1);
          unpack2(z23, z2, z3);
          Z = fmaf(Z, rs, (z0 + z1) + (z2 + z3));
          if (kEntropy) W = fmaf(W, rs, (wz[0] + wz[1]) + (wz[2] + wz[3]));
        };
        int j = 0;
        // Steady state: tiles that lie fully inside the cache are taken by both sub-tiles and need no mask, so the ring
        // position advances by two batches per tile and the loop carries no other bookkeeping.
        const int n_simple = (w.sub_valid[0] && w.sub_valid[1]) ? min(n / kTile, w.ntiles) : 0;
        // Lazy reference (kLazyMax): the exponentials of a steady-state tile are taken against the running reference
        // m_run AS IT STANDS -- no tile maximum, no rescale of Z -- which is exact as long as nothing overflows (fp32
        // sums are scale-free; m_run only has to stay within ~2^100 of the row maximum).  Each warp then votes on
        // "tile sum and Z finite and below 2^100"; a warp that fails (first tile of a row, or a jump of the maximum by
        // more than 100 in the log2 domain) discards its tile sums, re-reads the tile from tensor memory (the buffer is
        // released only after the vote) and takes the exact path, which also re-bases m_run and Z.
        for (; j < n_simple; ++j) {
          int own = buf + s, oph = ph;
          if (own >= kAccBufs) { own -= kAccBufs; oph ^= 1; }
          buf += 2;
          if (buf >= kAccBufs) { buf -= kAccBufs; ph ^= 1; }
          uint32_t v0[32], v1[32];
          if (!kLazyMax || kEntropy) {
            load_tile(own, oph, v0, v1);
            row_update(v0, v1, kHalf);
            continue;
          }
          mbar_wait(bar_sfull + 8 * own, oph);
          tc_fence_after();
          const uint32_t t_addr = t_col + (uint32_t)(own * kTile);
          tc_ld32(t_addr, v0);
          tc_ld32(t_addr + 32, v1);
          tc_wait_ld();
          // the polynomial exponentials are only valid up to 2^127 and, unlike the MUFU ones, do not overflow to inf:
          // their largest raw score takes part in the vote (c2 > 0)
          float pmax = -INFINITY;
#pragma unroll
          for (int pi = 0; pi < 32; ++pi)
            if (pair_is_poly(pi)) {
              const uint32_t* v = pi < 16 ? v0 : v1;
              pmax = fmaxf(pmax, fmaxf(__uint_as_float(v[(2 * pi) & 31]), __uint_as_float(v[(2 * pi + 1) & 31])));
            }
          uint64_t z01 = 0ull, z23 = 0ull;
          const uint64_t c2c2 = pack2(c2, c2), nm = pack2(-m_run, -m_run);
#pragma unroll
          for (int e = 0; e < 32; e += 4) {
            z01 = add2z(z01, ex2_pair(fma2(pack2u(v0[e], v0[e + 1]), c2c2, nm), e / 2));
            z23 = add2z(z23, ex2_pair(fma2(pack2u(v0[e + 2], v0[e + 3]), c2c2, nm), e / 2 + 1));
          }
#pragma unroll
          for (int e = 0; e < 32; e += 4) {
            z01 = add2z(z01, ex2_pair(fma2(pack2u(v1[e], v1[e + 1]), c2c2, nm), 16 + e / 2));
            z23 = add2z(z23, ex2_pair(fma2(pack2u(v1[e + 2], v1[e + 3]), c2c2, nm), 16 + e / 2 + 1));
          }
          float z0, z1, z2, z3;
          unpack2(z01, z0, z1);
          unpack2(z23, z2, z3);
          const float zt = (z0 + z1) + (z2 + z3);
          const bool ok = zt < 1.2676506e30f && Z < 1.2676506e30f &&   // 2^100; false for inf and NaN too
                          fmaf(pmax, c2, -m_run) < 100.f;
          if (__all_sync(0xffffffffu, ok)) {
            Z += zt;
          } else {
            tc_ld32(t_addr, v0);   // the fast path consumed the registers in place
            tc_ld32(t_addr + 32, v1);
            tc_wait_ld();
            row_update(v0, v1, kHalf);
          }
          tc_fence_before();
          __syncwarp();
          release(own);
        }
        // selects on the warp-uniform s, not dynamic indexing: a local-memory load would take the ring bookkeeping off the
        // uniform datapath (it did: +7 % cycles)
        const int ntp_mine = uniform(s == 0 ? w.ntp[0] : w.ntp[1]), ntp_other = uniform(s == 0 ? w.ntp[1] : w.ntp[0]);
        for (; j < w.ntiles; ++j) {   // last cache tile, chunk tiles (causal edge), sub-tiles of unequal length
          const bool tk_mine = j < ntp_mine, tk_other = j < ntp_other;   // the batches of tile j that exist (pair level)
          const bool tk0 = s == 0 ? tk_mine : tk_other, tk1 = s == 0 ? tk_other : tk_mine;
          if (s == 1 && tk0) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } }   // sub-tile 0's batch of tile j
          if (!(s == 0 ? tk0 : tk1)) { if (s == 0 && tk1) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } } continue; }
          // number of visible key columns of this tile for this row, relative to this thread's first column
          int limit;
          if (j < w.n_cache_tiles) limit = n - j * kTile;
          else {
            const int t0 = (j - w.n_cache_tiles) * kTile;
            limit = p.Nn - t0;
            if (p.causal) limit = min(limit, i - t0 + 1);
          }
          limit -= col0;
          uint32_t v0[32], v1[32];
          load_tile(buf, ph, v0, v1);
          if (++buf == kAccBufs) { buf = 0; ph ^= 1; }
          if (s == 0 && tk1) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } }    // sub-tile 1's batch of tile j
          row_update(v0, v1, limit);
        }
        // merge the two column halves of each row (online-softmax partials), then publish
        if (half == 1) sMg[s * kTile + r] = make_float4(m_run, Z, W, 0.f);
        named_bar_sync(1 + s, 256);
        if (half == 0) {
          const float4 o = sMg[s * kTile + r];
          const float m = fmaxf(m_run, o.x);
          const float r0 = ex2(m_run - m), r1 = ex2(o.x - m);
          Z = Z * r0 + o.y * r1;
          W = W * r0 + o.z * r1;
          // lse2 = log2 sum_k 2^(c2 s_k), stored negated; padded rows (i >= Nn) publish -inf so that pass 2 adds 2^-inf = 0
          const long long hq = (long long)w.lhA;
          const float l2 = m + log2f(Z);
          a.lse2[hq * a.lse_stride + i] = i < p.Nn ? -l2 : -INFINITY;  // stored NEGATED: pass 2 does one FMA
          if (i < p.Nn) {
            if (a.lse_nat) a.lse_nat[hq * p.Nn + i] = l2 * 0.6931471805599453f;
            if (kEntropy && a.row_entropy) a.row_entropy[hq * p.Nn + i] = (l2 - W / Z) * 0.6931471805599453f;
          }
        }
      } else {
        const int krow = w.rowA0 + s * kTile + r;  // key row in cache or chunk
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        uint64_t acc01 = 0ull, acc23 = 0ull;   // packed fp32x2 partial sums of the unmasked tiles
        const uint64_t c2c2 = pack2(c2, c2);
        const int it_first = w.seq0, it_end = w.seq0 + w.tiles_per_g;
        auto load_tile = [&](int b, int bph, uint32_t (&v0)[32], uint32_t (&v1)[32]) {
          mbar_wait(bar_sfull + 8 * b, bph);
          tc_fence_after();
          const uint32_t t_addr = t_col + (uint32_t)(b * kTile);
          tc_ld32(t_addr, v0);
          tc_ld32(t_addr + 32, v1);
          tc_wait_ld();
          tc_fence_before();
          __syncwarp();
          release(b);
        };
        // a_k += sum over this thread's 64 query columns of 2^(c2 s - lse2); every column visible
        auto col_update = [&](const uint32_t (&v0)[32], const uint32_t (&v1)[32], uint32_t l_addr) {
#pragma unroll
          for (int e4 = 0; e4 < 8; ++e4) {
            const float4 la = lds128(l_addr + e4 * 16), lb = lds128(l_addr + 128 + e4 * 16);
            const uint64_t x0 = fma2(pack2u(v0[4 * e4], v0[4 * e4 + 1]), c2c2, pack2(la.x, la.y));
            const uint64_t x1 = fma2(pack2u(v0[4 * e4 + 2], v0[4 * e4 + 3]), c2c2, pack2(la.z, la.w));
            const uint64_t x2 = fma2(pack2u(v1[4 * e4], v1[4 * e4 + 1]), c2c2, pack2(lb.x, lb.y));
            const uint64_t x3 = fma2(pack2u(v1[4 * e4 + 2], v1[4 * e4 + 3]), c2c2, pack2(lb.z, lb.w));
            acc01 = add2z(acc01, ex2_pair(x0, 4 * e4));
            acc23 = add2z(acc23, ex2_pair(x1, 4 * e4 + 1));
            acc01 = add2z(acc01, ex2_pair(x2, 4 * e4 + 2));
            acc23 = add2z(acc23, ex2_pair(x3, 4 * e4 + 3));
          }
        };
        // rescue: running reference mx and sum zl of 2^(x - mx) over this thread's columns, x = c2 s - lse2.  Masked columns
        // drop out, and so do weights below 2^-1074: fp64, the oracle's type, ends there (its psi jumps to 0 at that point).
        [[maybe_unused]] float mx = -1e30f, zl = 0.f;
        [[maybe_unused]] auto log_update = [&](const uint32_t (&v0)[32], const uint32_t (&v1)[32], uint32_t l_addr, int first) {
          float x[kHalf];
#pragma unroll
          for (int e4 = 0; e4 < 8; ++e4) {
            const float4 la = lds128(l_addr + e4 * 16), lb = lds128(l_addr + 128 + e4 * 16);
            const float le[8] = {la.x, la.y, la.z, la.w, lb.x, lb.y, lb.z, lb.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const float xa = fmaf(__uint_as_float(v0[4 * e4 + u]), c2, le[u]);
              const float xb = fmaf(__uint_as_float(v1[4 * e4 + u]), c2, le[4 + u]);
              x[4 * e4 + u] = (4 * e4 + u >= first && xa >= -1074.f) ? xa : -INFINITY;
              x[32 + 4 * e4 + u] = (32 + 4 * e4 + u >= first && xb >= -1074.f) ? xb : -INFINITY;
            }
          }
          float tm[4] = {x[0], x[1], x[2], x[3]};
#pragma unroll
          for (int e = 4; e < kHalf; ++e) tm[e & 3] = fmaxf(tm[e & 3], x[e]);
          const float m_new = fmaxf(mx, fmaxf(fmaxf(tm[0], tm[1]), fmaxf(tm[2], tm[3])));
          float zs[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int e = 0; e < kHalf; ++e) zs[e & 3] += ex2(x[e] - m_new);
          zl = fmaf(zl, ex2(mx - m_new), (zs[0] + zs[1]) + (zs[2] + zs[3]));
          mx = m_new;
        };
        if (kPass == 2 && w.sub_valid[0] && w.sub_valid[1] && !(p.causal && w.a_chunk)) {
          const SteadyState st = colsum_steady(w.ntiles, s, half, jt, t_col, c2, buf, ph, acc01, acc23);
          buf = st.buf; ph = st.ph; acc01 = st.acc01; acc23 = st.acc23;
        } else {
        int it_next = it_first;
        const int it0p_mine = uniform(s == 0 ? w.it0p[0] : w.it0p[1]), it0p_other = uniform(s == 0 ? w.it0p[1] : w.it0p[0]);
        const bool validp_mine = uniform(s == 0 ? w.validp[0] : w.validp[1]) != 0, validp_other = uniform(s == 0 ? w.validp[1] : w.validp[0]) != 0;
        for (int j = 0; j < w.ntiles; ++j) {
          const int it = it_next, slot = (jt + j) & (kLseSlots - 1), lse_parity = ((jt + j) / kLseSlots) & 1;   // kLseSlots is a power of two
          if (++it_next == it_end) it_next = it_first;                                       // no division in the tile loop
          const bool tk_mine = validp_mine && it >= it0p_mine, tk_other = validp_other && it >= it0p_other;   // pair level
          const bool tk0 = s == 0 ? tk_mine : tk_other, tk1 = s == 0 ? tk_other : tk_mine;
          const bool other = s == 0 ? tk1 : tk0;
          if (s == 1 && other) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } }   // sub-tile 0's batch of tile j comes first
          if (!(s == 0 ? tk0 : tk1)) { if (s == 0 && other) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } } continue; }
          // causal (R3): chunk key krow is visible to query i iff i >= krow; first visible column (thread-relative):
          const int first = ((p.causal && w.a_chunk) ? krow - it * kTile : 0) - col0;
          uint32_t v0[32], v1[32];
          load_tile(buf, ph, v0, v1);
          if (++buf == kAccBufs) { buf = 0; ph ^= 1; }
          if (s == 0 && other) { if (++buf == kAccBufs) { buf = 0; ph ^= 1; } }   // sub-tile 1's batch of tile j
          mbar_wait(bar_lse + 8 * slot, lse_parity);
          // one uniform register for the whole address (taken before the per-thread branch below): left to itself ptxas
          // keeps it as a sum of two uniform parts and materialises a vector copy of one of them for each of the 16 loads
          const uint32_t l_addr = (uint32_t)uniform((int)(sLse + (uint32_t)(slot * kTile + col0) * 4));
          if constexpr (kPass == 3) {
            log_update(v0, v1, l_addr, first);
          } else if (first <= 0) {
            col_update(v0, v1, l_addr);
          } else {
#pragma unroll
            for (int e4 = 0; e4 < 8; ++e4) {
              const float4 la = lds128(l_addr + e4 * 16), lb = lds128(l_addr + 128 + e4 * 16);
              const float le[8] = {la.x, la.y, la.z, la.w, lb.x, lb.y, lb.z, lb.w};
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const float pa = ex2(fmaf(__uint_as_float(v0[4 * e4 + u]), c2, le[u]));
                const float pb = ex2(fmaf(__uint_as_float(v1[4 * e4 + u]), c2, le[4 + u]));
                acc[u] += (4 * e4 + u >= first ? pa : 0.f) + (32 + 4 * e4 + u >= first ? pb : 0.f);
              }
            }
          }
        }
        }
        float q0, q1, q2, q3;
        unpack2(acc01, q0, q1);
        unpack2(acc23, q2, q3);
        const float part = ((acc[0] + acc[1]) + (acc[2] + acc[3])) + ((q0 + q1) + (q2 + q3));
        if (half == 1) {
          if constexpr (kPass == 3) sMg[s * kTile + r] = make_float4(mx, zl, 0.f, 0.f);
          else sMg[s * kTile + r].x = part;
        }
        named_bar_sync(1 + s, 256);
        const int n_v = p.n_v[w.l], n = p.n[w.l];
        const bool valid = w.a_chunk ? krow < p.Nn : krow < n;
        if (half == 0 && valid) {
          int m, t;
          if (w.a_chunk) chunk_row_to_seg(p, n_v, n, krow, m, t); else cache_row_to_seg(n_v, krow, m, t);
          float* out = m == 0 ? a.a_v + (long long)w.lhA * p.seg_cap_v : a.a_a + (long long)w.lhA * p.seg_cap_a;
          if constexpr (kPass == 3) {
            // only the keys pass 2 could not hold are replaced; finalize reads la for exactly those
            if (!(out[t] >= kTinyImportance)) {
              const float4 o = sMg[s * kTile + r];
              const float M = fmaxf(mx, o.x);
              const float Z = zl * ex2(mx - M) + o.y * ex2(o.x - M);
              const float la = Z > 0.f ? M + log2f(Z) : -INFINITY;
              (m == 0 ? a.la_v + (long long)w.lhA * p.seg_cap_v : a.la_a + (long long)w.lhA * p.seg_cap_a)[t] = la;
              out[t] = exp2f(la);   // what fp32 can hold of it (usually 0)
            }
          } else {
            out[t] = part + sMg[s * kTile + r].x;
          }
        }
        jt = (jt + w.ntiles) & (2 * kLseSlots - 1);
      }
    }
    if (idle_partner) named_bar_sync(3, 512);
    }  // work items
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(kTmemCols) : "memory");
  }
}

// natural-log LSE supplied by the caller -> internal log2-domain, padded layout
__global__ void lse_to_log2_kernel(const float* __restrict__ lse_nat, float* __restrict__ lse2, int rows, int Nn, int stride) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)rows * stride) return;
  const int i = (int)(idx % stride);
  const long long r = idx / stride;
  lse2[idx] = i < Nn ? -lse_nat[r * Nn + i] * 1.4426950408889634f : -INFINITY;
}

// Rescue, step 1: which of pass 2's items (256 stationary key rows of one (layer, KV head); same numbering as its item
// grid) hold a key that exists and whose fp32 column sum is below 2^-100.  One block per item, one thread per key row;
// flagged items are appended to `list` (order is irrelevant: every item's results are its own).
__global__ void __launch_bounds__(2 * kTile) rescue_items_kernel(const TcArgs a, int* __restrict__ list, int* __restrict__ count) {
  const StepParams& p = a.p;
  const int item = blockIdx.x;
  const int bx = item % a.nx, yz = item / a.nx, h = yz % a.ny, l = yz / a.ny;
  bool flag = false;
  if (!layer_skips_scoring(p, l)) {
    const int n_v = p.n_v[l], n = p.n[l];
    const bool in_chunk = bx >= a.n_cache_pairs;
    const int krow = (in_chunk ? bx - a.n_cache_pairs : bx) * 2 * kTile + threadIdx.x;
    if (krow < (in_chunk ? p.Nn : n)) {
      int m, t;
      if (in_chunk) chunk_row_to_seg(p, n_v, n, krow, m, t); else cache_row_to_seg(n_v, krow, m, t);
      const long long lh = (long long)l * p.Hkv + h;
      flag = !((m == 0 ? a.a_v + lh * p.seg_cap_v : a.a_a + lh * p.seg_cap_a)[t] >= kTinyImportance);
    }
  }
  if (__syncthreads_or(flag) && threadIdx.x == 0) list[atomicAdd(count, 1)] = item;
}

// ---- host side -------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static cudaError_t get_encode(omnimem_ctx* ctx, EncodeTiledFn* fn) {
  if (!ctx->encode_tiled) {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q);
    if (e != cudaSuccess) return e;
    if (q != cudaDriverEntryPointSuccess || !f) return cudaErrorNotSupported;
    ctx->encode_tiled = f;
  }
  *fn = (EncodeTiledFn)ctx->encode_tiled;
  return cudaSuccess;
}

// [outer, rows, 128] bf16 row-major -> 3-D map, box = 64 x 128 x 1, 128-byte swizzle, zero fill out of bounds
static cudaError_t make_map(EncodeTiledFn enc, CUtensorMap* m, const void* base, uint64_t rows, uint64_t outer) {
  if (rows == 0 || outer == 0 || base == nullptr) { memset(m, 0, sizeof(*m)); return cudaSuccess; }
  const cuuint64_t dims[3] = {(cuuint64_t)kHeadDim, rows, outer};
  const cuuint64_t strides[2] = {(cuuint64_t)kHeadDim * 2, rows * kHeadDim * 2};
  const cuuint32_t box[3] = {(cuuint32_t)kKBlock, (cuuint32_t)kTile, 1};
  const cuuint32_t es[3] = {1, 1, 1};
  const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

struct Maps { CUtensorMap q, kc, kn; };

static cudaError_t make_maps(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, Maps* m) {
  EncodeTiledFn enc;
  cudaError_t e = get_encode(const_cast<omnimem_ctx*>(ctx), &enc);
  if (e != cudaSuccess) return e;
  if ((e = make_map(enc, &m->q, b.Q, p.Nn, (uint64_t)p.L * p.Hq)) != cudaSuccess) return e;
  if ((e = make_map(enc, &m->kc, b.cacheK, p.cache_cap, (uint64_t)p.L * p.Hkv)) != cudaSuccess) return e;
  return make_map(enc, &m->kn, b.chunkK, p.Nn, (uint64_t)p.L * p.Hkv);
}

static TcArgs make_args(const StepParams& p, const StepBuffers& b) {
  TcArgs a{};
  a.p = p;
  a.lse2 = b.lse2;
  a.lse_stride = (p.Nn + kTile - 1) / kTile * kTile;
  a.lse_nat = b.lse_out;
  a.row_entropy = b.row_entropy;
  a.a_v = b.a_v;
  a.a_a = b.a_a;
  a.n_cache_pairs = (p.cache_cap + 2 * kTile - 1) / (2 * kTile);
  return a;
}

// One launch of a scoring kernel: persistent CTAs (one per SM, 210 KB of dynamic shared memory each) that draw the
// nx * ny * nz work items from a device counter, which is zeroed on the stream right before the launch.
typedef void (*ScoreKernel)(const CUtensorMap, const CUtensorMap, const CUtensorMap, const TcArgs);
static cudaError_t launch_score(const omnimem_ctx* ctx, ScoreKernel k, dim3 items, int which, cudaStream_t st, const Maps& m, TcArgs a) {
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return e;
  a.nx = (int)items.x;
  a.ny = (int)items.y;
  a.n_items = (int)(items.x * items.y * items.z);
  a.counter = ctx->sched + which;
  if ((e = cudaMemsetAsync(a.counter, 0, sizeof(int), st)) != cudaSuccess) return e;
  const int ctas = ctx->cfg.score_ctas > 0 && ctx->cfg.score_ctas < ctx->sm_count ? ctx->cfg.score_ctas : ctx->sm_count;
  const int grid = a.n_items < ctas ? a.n_items : ctas;
  k<<<grid, kThreads, kSmemBytes, st>>>(m.q, m.kc, m.kn, a);
  return cudaGetLastError();
}

cudaError_t launch_lse_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches) {
  if (p.Nn == 0) return cudaSuccess;
  Maps m;
  cudaError_t e = make_maps(ctx, p, b, &m);
  if (e != cudaSuccess) return e;
  const TcArgs a = make_args(p, b);
  dim3 grid((p.Nn + 2 * kTile - 1) / (2 * kTile), p.Hq, p.L);
  ++*launches;
  if (b.row_entropy) return launch_score(ctx, score_tc_kernel<1, true>, grid, 0, st, m, a);
  return launch_score(ctx, score_tc_kernel<1, false>, grid, 0, st, m, a);
}

cudaError_t launch_colsum_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches) {
  if (p.Nn == 0) {  // no queries: a = 0 everywhere
    cudaError_t e = cudaMemsetAsync(b.a_v, 0, (size_t)p.L * p.Hkv * p.seg_cap_v * sizeof(float), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(b.a_a, 0, (size_t)p.L * p.Hkv * p.seg_cap_a * sizeof(float), st);
    return e;
  }
  Maps m;
  cudaError_t e = make_maps(ctx, p, b, &m);
  if (e != cudaSuccess) return e;
  const TcArgs a = make_args(p, b);
  if (b.lse_in) {
    const long long tot = (long long)p.L * p.Hq * a.lse_stride;
    lse_to_log2_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(b.lse_in, b.lse2, p.L * p.Hq, p.Nn, a.lse_stride);
    ++*launches;
  }
  dim3 grid(a.n_cache_pairs + (p.Nn + 2 * kTile - 1) / (2 * kTile), p.Hkv, p.L);
  ++*launches;
  return launch_score(ctx, score_tc_kernel<2, false>, grid, 1, st, m, a);
}

// Eq.6 below fp32's range on the tensor-core path (R31): flag the items, then redo exactly those in the log domain.
// rescue_items: [1 + items] ints of scratch (count, then the list).  Worst case (every item flagged) = one more pass over
// Q K^T on the tensor cores; nothing flagged = one sweep over a and a kernel whose CTAs find an empty list.
cudaError_t launch_colsum_rescue_tc(const omnimem_ctx* ctx, const StepParams& p, const StepBuffers& b, cudaStream_t st, int* launches) {
  if (p.Nn == 0) return cudaSuccess;
  Maps m;
  cudaError_t e = make_maps(ctx, p, b, &m);
  if (e != cudaSuccess) return e;
  TcArgs a = make_args(p, b);
  a.la_v = b.la_v;
  a.la_a = b.la_a;
  const dim3 grid(a.n_cache_pairs + (p.Nn + 2 * kTile - 1) / (2 * kTile), p.Hkv, p.L);   // pass 2's item grid
  a.nx = (int)grid.x;
  a.ny = (int)grid.y;
  a.n_items = (int)(grid.x * grid.y * grid.z);
  int* count = b.rescue_items;
  int* list = b.rescue_items + 1;
  if ((e = cudaMemsetAsync(count, 0, sizeof(int), st)) != cudaSuccess) return e;
  rescue_items_kernel<<<a.n_items, 2 * kTile, 0, st>>>(a, list, count);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  a.item_list = list;
  a.item_count = count;
  *launches += 2;
  return launch_score(ctx, score_tc_kernel<3, false>, grid, 3, st, m, a);
}

}  // namespace omnimem
