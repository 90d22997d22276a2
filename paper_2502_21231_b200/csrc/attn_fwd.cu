// attn_fwd.cu — bs_attn_fwd: one Q-chunk x KV-chunk step of packed varlen / zigzag-CP causal
// attention on sm_100a (SURVEY.md 8(a) a2+a3; flash attention = exact attention).
//
// Kernel shape: one persistent CTA per SM, 640 threads at 96 registers, 1 CTA / SM:
//   warps 0-15  softmax: warpgroup g = warp / 4 works on Q tile t = g / 2, key columns
//               [64 hf, 64 hf + 64) of every block with hf = g % 2 - two threads share a row (row r
//               of the tile <-> threads r and 128 + r of the tile's 256), the row maximum and the
//               row sum are exchanged through shared memory
//   warp  16/18 MMA issuers of Q tile 0 / 1 (one elected lane each): tcgen05.mma, accumulators in
//               TMEM; a turn lock keeps the two tiles' batches half a period apart
//   warp  17    lane 0: TMA producer (Q per unit and tile, K/V blocks through a 4-stage ring, the
//               accumulator-clearing stores)
//   warp  19    scheduler (sched.cuh): pulls units from the global cursor into a shared-memory ring
// A work item is (up to 256 query rows = two 128-row tiles of one query range, one query head).
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,256+D) O1 [384,384+D); P (bf16) of 16 keys
// overwrites the first 8 of the 16 S columns of those keys.  Per tile the chain is S(b) -> softmax
// -> P(b) -> PV(b), S(b+1); the two tiles run it independently, so the softmax of one overlaps
// the MMAs of the other, and P is handed over in four 16-column chunks (order 3, 2, 0, 1) so that
// PV starts under the remaining exponentials.  Softmax is fp32 with exp2, a lazily updated
// running max (O is rescaled only when the max grew by more than 2^8) and the row sum kept in
// fp32; O is normalised and written as bf16 with LSE = m ln2 + ln l at the end.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include <type_traits>

#include "common.h"
#include "launch_utils.h"
#include "ptx.cuh"
#include "sched.cuh"
#include "worklist.h"

#define BS_TRACE_KERNEL_FWD
#include "trace.cuh"

namespace {

using namespace bs;
using namespace bs::ptx;

#ifndef BS_SCHED_SLOTS
#define BS_SCHED_SLOTS 2
#endif
constexpr int kFwdSchedSlots = BS_SCHED_SLOTS;  // depth of the scheduler ring (sched.cuh)
using SchedRing = SchedRingT<kFwdSchedSlots>;
using UnitProducer = UnitProducerT<kFwdSchedSlots>;
using UnitConsumer = UnitConsumerT<kFwdSchedSlots>;
constexpr int kSchedRingBytes = SchedRing::kBytes;

constexpr int kFwdThreads = 640;      // 4 softmax warpgroups + 1 auxiliary warpgroup (MMA, TMA)
constexpr int kMmaWarp0 = 16, kTmaWarp = 17, kSchedWarp = 19;  // warps 16 / 18 issue the MMAs of Q tile 0 / 1
constexpr int kRegsSoftmax = 104;     // setmaxnreg: 512 * 104 + 128 * 96 = 65536 (compiled at 96)
constexpr int kStages = 4;              // K/V ring depth (K and V blocks alternate in the ring)
constexpr float kRescaleThreshold = 8.f;  // log2 units
#ifndef BS_FWD_EMU
#define BS_FWD_EMU 1
#endif
constexpr int kEmuOf4 = BS_FWD_EMU;  // of every 4 column pairs, this many take the FMA-pipe exp2

struct FwdParams {
  SchedView sv;     // units = query items x n_q_heads
  int32_t n_q_heads, group;  // group = Hq / Hkv
  int32_t q_rows;
  float scale_log2;  // softmax_scale * log2(e)
  __nv_bfloat16* O;
  float* LSE;
  int64_t o_row_stride, lse_head_stride;
  int32_t wide_stores;  // O rows are 32-byte aligned: 256-bit stores in the epilogue
  int32_t clear_acc;  // also zero the fp32 dQ accumulator rows of every unit (TMA stores of zeros)
};

template <int D>
struct FwdSmem {
  static constexpr int kTileBytes = kTile * D * 2;  // one 128-row tile of Q, K or V
  static constexpr int kQOff = 0;                   // 2 Q tiles
  static constexpr int kKVOff = 2 * kTileBytes;     // kStages K/V tiles
  static constexpr int kBarOff = kKVOff + kStages * kTileBytes;
  // barriers: q_full[2], q_empty[2], kv_full[S], kv_empty[S], s_full[2], p_full[2][4], o_full[2]
  static constexpr int kNumBars = 4 + 2 * kStages + 12;
  static constexpr int kTmemSlotOff = kBarOff + kNumBars * 8;
  static constexpr int kSchedOff = kTmemSlotOff + 16;  // SchedRing of the dynamic scheduler
  static constexpr int kXchOff = kSchedOff + kSchedRingBytes;     // row max [2 tiles][2][2][128], row sum [2][2][128]
  static constexpr int kLockOff = kXchOff + 6144;     // turn lock of the two MMA issuers
  static constexpr int kZeroOff = ((kLockOff + 16 + 127) / 128) * 128;  // 8 KB of zeros (TMA source)
  static constexpr int kBytes = kZeroOff + 8192;
  static constexpr int kAlloc = kBytes + 1024;  // slack to align the base to 1024 B
};

// Per-tile block count of one span: number of 128-key blocks with at least one visible pair.
// at0 = local index of the tile's first row, rows = valid rows of the tile.
__device__ __forceinline__ int span_blocks(int at0, int rows, const Span& sp) {
  if (rows <= 0) return 0;
  const int vis = min(sp.len, at0 + rows - 1 + sp.off + 1);
  return vis > 0 ? (vis + kTile - 1) / kTile : 0;
}


// Walks the 128-key blocks of an item in (span, block) order.  A block is visited if either Q
// tile has a visible pair in it; tile t takes part in the block iff active(t).  (Scalar members
// only: arrays indexed by the runtime tile number would live in local memory.)
template <bool kUniform>
struct WalkerT {
  const Span* table;
  const Unit* u;
  int n_spans, s, j, nb0, nb1, at0_1, rows0, rows1;
  int flip;  // TMEM / shared-memory slot t works on Q tile t ^ flip of the item (see tile())
  Span sp;
  // The upper tile of a causal pair visits one block more than the lower one.  With a fixed
  // assignment the slot of the lower tile runs ahead by a block per unit until the K/V ring stops
  // it, and from then on every stage is held for the trailing slot: no prefetch distance left.
  // Alternating the assignment from unit to unit keeps the two slots within one block (a rule
  // on the blocks given to each slot so far alternates the same way and measured no better).
  __device__ __forceinline__ int tile(int t) const { return t ^ flip; }
  __device__ __forceinline__ int at0(int t) const { return tile(t) ? at0_1 : at0_1 - kTile; }
  __device__ __forceinline__ int rows(int t) const { return tile(t) ? rows1 : rows0; }
  __device__ __forceinline__ void load_span() {
    while (s < n_spans) {
      sp = unit_span(*u, table, s);
      if (kUniform) {  // converged warp, same span in every lane
        sp.begin = warp_uniform(sp.begin);
        sp.len = warp_uniform(sp.len);
        sp.off = warp_uniform(sp.off);
      }
      nb0 = span_blocks(at0_1 - kTile, rows0, sp);
      nb1 = span_blocks(at0_1, rows1, sp);
      if (max(nb0, nb1) > 0) break;
      ++s;
    }
    j = 0;
  }
  __device__ __forceinline__ void init(const Span* sp_table, const Unit& unit, int flip_) {
    const Item& it = unit.item;
    flip = flip_;
    table = sp_table;
    u = &unit;
    n_spans = it.n_spans;
    at0_1 = it.local0 + kTile;
    rows0 = max(0, min(kTile, it.range_len - it.local0));
    rows1 = max(0, min(kTile, it.range_len - at0_1));
    s = 0;
    load_span();
  }
  __device__ __forceinline__ bool done() const { return s >= n_spans; }
  __device__ __forceinline__ bool active(int t) const { return j < (tile(t) ? nb1 : nb0); }
  __device__ __forceinline__ void next() {
    if (++j >= max(nb0, nb1)) {
      ++s;
      load_span();
    }
  }
  // total blocks tile t takes part in over the whole item (counted by the host: the loop over
  // the spans cost the MMA issuer ~1500 cycles in front of every unit's first S MMA)
  __device__ __forceinline__ int total(int t) const {
    return tile(t) ? u->item.tile_blocks[1] : u->item.tile_blocks[0];
  }
};
using Walker = WalkerT<false>;

template <int D>
__device__ __forceinline__ void issue_qk(uint32_t tmem_s, uint32_t q_addr, uint32_t k_addr) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, kTile, 0, 0);
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk) {
    const uint32_t o = (kk / 4) * (kTile * 128) + (kk % 4) * 32;  // 64-column box, 16 columns = 32 B
    umma_ss(tmem_s, umma_desc_sw128(q_addr + o, 16, 1024), umma_desc_sw128(k_addr + o, 16, 1024),
            idesc, kk > 0);
  }
}
// O (+)= P V for the 2 x 16 keys of one chunk slot: the softmax threads of both column halves
// produce their 16-column chunks in the order 3, 2, 0, 1 and hand each over separately, so that
// the first PV MMAs run under the remaining exponentials.
__device__ __forceinline__ int chunk_of_slot(int slot) { return (0x3201 >> (4 * (3 - slot))) & 3; }
template <int D>
__device__ __forceinline__ void issue_pv_slot(uint32_t tmem_o, uint32_t tmem_p, uint32_t v_addr,
                                              int slot, bool accumulate) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, D, 0, 1);  // B = V is MN-major (d contiguous)
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int kk = half * 4 + chunk_of_slot(slot);
    // 16 keys = 16 rows of 128 B; the second 64-wide d half (D = 128) is one box (16 KB) further
    // P of keys [16 kk, 16 kk + 16) sits over the first 8 columns of its own 16 S columns
    umma_ts(tmem_o, tmem_p + kk * 16, umma_desc_sw128(v_addr + kk * 2048, kTile * 128, 1024), idesc,
            accumulate || half > 0);
  }
}

}  // namespace

namespace {

struct Ring {  // position in the K/V smem ring
  uint32_t stage = 0, phase = 0;
  __device__ __forceinline__ void advance() {
    if (++stage == kStages) {
      stage = 0;
      phase ^= 1;
    }
  }
};

template <int D>
__global__ void __launch_bounds__(kFwdThreads, 1)
attn_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmZ,
                const __grid_constant__ FwdParams p) {
  using L = FwdSmem<D>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) &
                                             ~uintptr_t(1023));
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOff);
  uint64_t* q_full = bars;       // [2] per Q tile
  uint64_t* q_empty = bars + 2;  // [2]
  uint64_t* kv_full = bars + 4;
  uint64_t* kv_empty = bars + 4 + kStages;
  uint64_t* s_full = bars + 4 + 2 * kStages;
  uint64_t* p_full = s_full + 2;  // [tile][chunk slot]
  uint64_t* o_full = p_full + 8;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kTmemSlotOff);
  SchedRing* sched = reinterpret_cast<SchedRing*>(smem + L::kSchedOff);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == kTmaWarp && lane == 0) {
    *reinterpret_cast<uint32_t*>(smem + L::kLockOff) = 0;
    sched_ring_init(sched, 4 * kTile / 32 + 3);  // 16 softmax warps + 2 MMA lanes + the TMA lane
    for (int t = 0; t < 2; ++t) {
      mbar_init(&q_full[t], 1);
      mbar_init(&q_empty[t], 1);
      mbar_init(&s_full[t], 1);
      for (int c = 0; c < 4; ++c) mbar_init(&p_full[4 * t + c], 8);  // one arrival per softmax warp
      mbar_init(&o_full[t], 1);
    }
    for (int i = 0; i < kStages; ++i) {
      mbar_init(&kv_full[i], 1);
      mbar_init(&kv_empty[i], 2);  // both MMA issuers release a stage
    }
    fence_barrier_init();
    prefetch_tensormap(&tmQ);
    prefetch_tensormap(&tmK);
    prefetch_tensormap(&tmV);
  }
  if (p.clear_acc) {  // the zero source of the accumulator-clearing stores
    for (int i = threadIdx.x; i < 8192 / 16; i += blockDim.x)
      reinterpret_cast<uint4*>(smem + L::kZeroOff)[i] = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
  }
  if (warp == kMmaWarp0) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t smem_q = smem_u32(smem + L::kQOff), smem_kv = smem_u32(smem + L::kKVOff);

  if (warp >= kMmaWarp0) {
    if (warp == kTmaWarp && lane == 0) {
      // ===================================== TMA producer =====================================
      uint32_t q_ph[2] = {0, 0};
      uint64_t fenced = 0;  // clipped tensor maps (index < 64) this thread has fenced
      Ring ring;
      UnitConsumer cons{sched};
      Unit u;
      int un = -1;
      while (cons.next(&u)) {
        ++un;
        UTRACE(4, 0, un);
        const Item& it = u.item;
        const int h = u.head, g = h / p.group;
        if (p.clear_acc) {  // 256 rows x D fp32 of this (unit, head): 64-row x 32-column boxes
          for (int k = 0; k < 4; ++k)
            for (int c = 0; c < D / 32; ++c)
              tma_store_3d(&tmZ, smem + L::kZeroOff, c * 32, h, it.row0 + 64 * k);
          bulk_commit_group();
        }
        Walker wk;
        wk.init(p.sv.spans, u, un & 1);
        if (wk.done()) continue;
        // Order of a unit's loads: K of the first block (its ring stage is released early, at
        // the S MMAs four stages back), then the two Q tiles (a tile's buffer is released at its
        // last S MMA of the previous unit), then V of the first block and the rest.  V stages are
        // only released at PV MMAs, i.e. late in the previous unit: nothing S(0) needs may queue
        // behind them.
        // The V block that runs past the end of its key range is loaded through a tensor map whose
        // row extent ends at the range end (host-built, in the workspace), so that TMA zero-fills
        // the rows past it: a whole 128-row box through the buffer-wide map would bring in whatever
        // follows in the caller's buffer (another document, or uninitialised rows with NaN / Inf),
        // and P = 0 times NaN inside the PV contraction would poison every row of O.  A tensor map
        // in global memory must be fenced by the thread that uses it (~360 cycles): once per map
        // and CTA (bit mask; maps beyond the 64th are fenced at every use).
        auto load_kv = [&](int krow, const CUtensorMap* m, int clip) {
          if (clip >= 0 && (clip >= 64 || !((fenced >> clip) & 1))) {
            tensormap_acquire(m);
            if (clip < 64) fenced |= 1ull << clip;
          }
          mbar_wait(&kv_empty[ring.stage], ring.phase ^ 1);
          mbar_arrive_expect_tx(&kv_full[ring.stage], L::kTileBytes);
          for (int half = 0; half < D / 64; ++half)
            tma_load_3d(smem + L::kKVOff + ring.stage * L::kTileBytes + half * (kTile * 128), m,
                        &kv_full[ring.stage], half * 64, g, krow);
          ring.advance();
        };
        for (bool first = true; !wk.done(); wk.next(), first = false) {
          const int krow = wk.sp.begin + wk.j * kTile;
          load_kv(krow, &tmK, -1);
          if (first) {
            UTRACE(4, 1, un);
            for (int t = 0; t < 2; ++t) {
              if (wk.total(t) == 0) continue;
              mbar_wait(&q_empty[t], q_ph[t] ^ 1);
              UTRACE(4, 2 + t, un);
              q_ph[t] ^= 1;
              mbar_arrive_expect_tx(&q_full[t], L::kTileBytes);
              for (int half = 0; half < D / 64; ++half)
                tma_load_3d(smem + L::kQOff + t * L::kTileBytes + half * (kTile * 128), &tmQ,
                            &q_full[t], half * 64, h, it.row0 + wk.tile(t) * kTile);
            }
          }
          const int clip = (wk.sp.clip >= 0 && wk.sp.len - wk.j * kTile < kTile) ? wk.sp.clip : -1;
          load_kv(krow, clip >= 0 ? p.sv.tmaps + clip : &tmV, clip);
          if (first) UTRACE(4, 4, un);
        }
        UTRACE(4, 5, un);
      }
      if (p.clear_acc) bulk_wait_group<0>();  // the zero stores have landed before the CTA exits
    } else if (warp == kSchedWarp && lane == 0) {
      // ====================================== scheduler ======================================
      UnitProducer prod{sched};
      Unit u;
      while (prod.next(p.sv, &u)) {
      }
    } else if ((warp == kMmaWarp0 || warp == kMmaWarp0 + 2) && elect_one()) {
      // ============================ MMA issuer of Q tile t = 0 / 1 ============================
      // Each tile has its own issuing warp (one lane).
      const int t = (warp - kMmaWarp0) >> 1;
      const uint32_t tS = tmem + t * kTile, tO = tmem + 256 + t * kTile;
      const uint32_t sQ = smem_q + t * L::kTileBytes;
      uint32_t q_ph = 0, p_ph = 0;
      uint32_t* turn = reinterpret_cast<uint32_t*>(smem + L::kLockOff);
      int tr_it = 0;
      Ring ring;
      UnitConsumer cons{sched};
      Unit u;
      int un = -1;
      while (cons.next(&u)) {
        ++un;
        UTRACE(2 + t, 0, un);
        Walker cur;
        cur.init(p.sv.spans, u, un & 1);
        if (cur.done()) continue;
        const int tot = cur.total(t);
        UTRACE(2 + t, 1, un);
        int n_s = 0, n_pv = 0;
        auto wait_q = [&]() {  // never called with the turn lock held
          if (n_s == 0) {
            mbar_wait(&q_full[t], q_ph);
            q_ph ^= 1;
            tc_fence_after();
          }
        };
        // S_t = Q_t K^T of one block; the last one of a unit releases the tile's Q buffer to the
        // producer (the next unit's Q streams in early)
        auto issue_s = [&](uint32_t k_stage) {
          ++n_s;
          {
            issue_qk<D>(tS, sQ, smem_kv + k_stage * L::kTileBytes);
            tc_commit(&s_full[t]);
            if (n_s == tot) tc_commit(&q_empty[t]);
          }
        };
        auto release = [&](uint32_t stage) {
          tc_commit(&kv_empty[stage]);
        };
        // prologue: S_t(0).  Every ring stage is waited for and released by both issuers, also
        // for blocks their tile takes no part in.
        mbar_wait(&kv_full[ring.stage], ring.phase);
        UTRACE(2 + t, 2, un);
        tc_fence_after();
        if (cur.active(t)) {
          wait_q();
          UTRACE(2 + t, 3, un);
          issue_s(ring.stage);
          UTRACE(2 + t, 4, un);
        }
        release(ring.stage);
        ring.advance();
        while (true) {
          Walker nxt = cur;
          nxt.next();
          const bool has_next = !nxt.done();
          const uint32_t v_stage = ring.stage;
          mbar_wait(&kv_full[ring.stage], ring.phase);
          ring.advance();
          const uint32_t k_stage = ring.stage;
          if (has_next) {
            mbar_wait(&kv_full[ring.stage], ring.phase);
            ring.advance();
          }
          tc_fence_after();
          if (cur.active(t)) {
            ++n_pv;
            // the first three chunk slots of P go to the tensor pipe as they arrive, outside the
            // turn lock (PV MMAs of one tile may interleave freely with the other tile's batch)
            for (int slot = 0; slot < 3; ++slot) {
              mbar_wait_spin(&p_full[4 * t + slot], p_ph);
              tc_fence_after();
              issue_pv_slot<D>(tO, tS, smem_kv + v_stage * L::kTileBytes, slot, n_pv > 1 || slot > 0);
            }
            mbar_wait_spin(&p_full[4 * t + 3], p_ph);
            p_ph ^= 1;
            if (lane == 0) TRACE(2 + t, 0, tr_it);
            tc_fence_after();
          }
          if (has_next && nxt.active(t)) wait_q();
          // The batch [PV_t(b), S_t(b+1)] is issued under the turn lock: batches of the two tiles
          // enter the tensor pipe whole, one after the other, which keeps the tiles half a period
          // apart (softmax of one under the MMAs of the other) instead of drifting into phase.
          while (atom_cas_shared(turn, 0u, 1u) != 0u) __nanosleep(20);
          if (lane == 0) TRACE(2 + t, 1, tr_it);
          if (cur.active(t)) {
            {
              issue_pv_slot<D>(tO, tS, smem_kv + v_stage * L::kTileBytes, 3, true);
              if (n_pv == tot) tc_commit(&o_full[t]);
            }
              if (lane == 0) TRACE(2 + t, 2, tr_it);
          }
          release(v_stage);
          if (has_next) {
            if (nxt.active(t)) issue_s(k_stage);
            release(k_stage);
          }
          if (lane == 0) TRACE(2 + t, 3, tr_it);
          st_release_shared(turn, 0u);
          if (lane == 0) TRACE(2 + t, 4, tr_it);
          ++tr_it;
          if (!has_next) break;
          cur = nxt;
        }
        UTRACE(2 + t, 5, un);
      }
    }
  } else {
    // ================================== softmax warpgroups ==================================
    // Warpgroup g = warp / 4 works on Q tile t = g / 2, key columns [64 hf, 64 hf + 64) with
    // hf = g % 2: two threads share a row (the row maximum and the row sum are exchanged through
    // shared memory), which halves the latency of the S -> P step that the MMAs wait for.
    // (no setmaxnreg: the kernel is compiled for 96 registers per thread, 640 * 96 = 61440)
    const int t = warp >> 3, hf = (warp >> 2) & 1;
    const int r = threadIdx.x & 127;    // row of the tile owned by this thread
    const uint32_t lane_addr = uint32_t((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + lane_addr + t * kTile + hf * 64;         // this half of S_t
    const uint32_t tO = tmem + lane_addr + 256 + t * kTile + hf * (D / 2);  // this half of O_t
    float* xch_m = reinterpret_cast<float*>(smem + L::kXchOff) + t * 512 + r;  // [parity][half][row]
    float* xch_l = reinterpret_cast<float*>(smem + L::kXchOff) + 1024 + t * 256 + r;  // [half][row]
    const float2 sc2 = make_float2(p.scale_log2, p.scale_log2);
    uint32_t s_ph = 0, o_ph = 0;
    int tr_it = 0;
    UnitConsumer cons{sched};
    Unit u;
    int un = -1;
    while (cons.next_warp(&u, 0xffffffffu, 0)) {
      ++un;
      if (r == 0 && hf == 0) UTRACE(t, 0, un);
      const Item& it = u.item;
      const int h = u.head;
      Walker wk;
      wk.init(p.sv.spans, u, un & 1);
      const int at0 = wk.at0(t);
      const bool valid = r < wk.rows(t);
      const int64_t grow = (int64_t)it.row0 + wk.tile(t) * kTile + r;
      __nv_bfloat16* o_ptr = p.O + grow * p.o_row_stride + (int64_t)h * D + hf * (D / 2);
      const int tot = wk.total(t);
      if (tot == 0) {  // no key of this call is visible to any row of the tile
        if (valid) {
          for (int c = 0; c < D / 16; ++c) reinterpret_cast<uint4*>(o_ptr)[c] = make_uint4(0, 0, 0, 0);
          if (hf == 0) p.LSE[(int64_t)h * p.lse_head_stride + grow] = -CUDART_INF_F;
        }
        continue;
      }
      float m_used = -CUDART_INF_F;
      float2 l2 = make_float2(0.f, 0.f);
      int cnt = 0;
      for (; !wk.done(); wk.next()) {
        if (!wk.active(t)) continue;
        mbar_wait(&s_full[t], s_ph);
        s_ph ^= 1;
        if (r == 0) TRACE(t, 0, tr_it);
        if (r == 0 && hf == 0 && cnt == 0) UTRACE(t, 1, un);
        tc_fence_after();
        // Two passes over this thread's 64 columns in chunks of 16, double-buffered in A / B so
        // that the TMEM load of the next chunk runs under the arithmetic of the current one.
        // Pass 1: row maximum.  Pass 2 (chunks 3, 2, 0, 1; chunk 3 is still in B): P = 2^(S c - m),
        // packed to bf16 and written over the chunk's own first 8 columns.
        const int b0 = wk.j * kTile;
        const bool edge_block = b0 + kTile - 1 > at0 + wk.sp.off || b0 + kTile > wk.sp.len;
        // The block body exists twice: interior blocks (all columns visible) run branch-free
        // straight-line code (the instruction fetch of a warp that jumps over the masking code
        // of every chunk costs 8 % of the kernel), blocks on a mask boundary the general one.
        auto softmax_block = [&](auto edge_c) {
        constexpr bool edge = decltype(edge_c)::value;
        // last visible column of this row relative to this thread's first column (>= 63: all)
        const int lim = edge ? min(at0 + r + wk.sp.off, wk.sp.len - 1) - b0 - hf * 64 : 64;
        // The same for the first and the last row of this warp (lim grows with the row): a chunk
        // is classified for the whole warp - every row sees all of it / no row sees any of it /
        // mixed - so that the rows of a warp never take different paths.
        const int lim_lo = edge ? __shfl_sync(0xffffffffu, lim, 0) : 64;
        const int lim_hi = edge ? __shfl_sync(0xffffffffu, lim, 31) : 64;
        float A[16], B[16];
        float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
        auto max16 = [&](const float* v) {
#pragma unroll
          for (int c = 0; c < 16; c += 4) {
            mx0 = fmax3(mx0, v[c], v[c + 1]);
            mx1 = fmax3(mx1, v[c + 2], v[c + 3]);
          }
        };
        // Pass 1: maximum over the visible columns.  It has to be exact: with an inflated
        // maximum the largest P of a row is no longer exactly 1, its bf16 rounding no longer
        // cancels against the fp32 row sum, and rows with few visible keys (the first rows of a
        // document) lose up to 2^-9 relative in O.  Chunks no row of the warp sees are skipped,
        // chunks every row sees take the plain code, only mixed chunks pay for selects.
        auto max16m = [&](const float* v, int k16) {
          const int lim_k = lim - k16;
          if (!edge || lim_lo - k16 >= 15) {
            max16(v);
          } else if (lim_hi - k16 >= 0) {
#pragma unroll
            for (int c = 0; c < 16; ++c) mx0 = fmaxf(mx0, c <= lim_k ? v[c] : -CUDART_INF_F);
          }
        };
        tmem_ld16(tS, reinterpret_cast<uint32_t*>(A));
        tmem_ld16(tS + 16, reinterpret_cast<uint32_t*>(B));
        tmem_wait_ld();
        max16m(A, 0);
        tmem_ld16(tS + 32, reinterpret_cast<uint32_t*>(A));
        max16m(B, 16);
        tmem_ld16(tS + 48, reinterpret_cast<uint32_t*>(B));
        tmem_wait_ld();
        max16m(A, 32);
        max16m(B, 48);  // chunk 3 stays in B for pass 2
        if (r == 0) TRACE(t, 1, tr_it);
        const float mx_half = fmaxf(mx0, mx1);
        // exchange the half-row maxima (slots alternate with the block parity; one barrier/block)
        xch_m[(cnt & 1) * 256 + hf * 128] = mx_half;
        bar_sync(1 + t, 2 * kTile);
        const float mx = fmaxf(mx_half, xch_m[(cnt & 1) * 256 + (hf ^ 1) * 128]) * p.scale_log2;
        const bool grow_max = mx > m_used + kRescaleThreshold;
        float alpha = 1.f;
        if (grow_max) {
          alpha = ex2(m_used - mx);  // 0 when nothing was visible so far
          m_used = mx;
          l2.x *= alpha;
          l2.y *= alpha;
        }
        if (cnt > 0 && __any_sync(0xffffffffu, grow_max)) {
          // S_t(b) complete implies PV_t(b-1) complete (issue order): O_t is stable here
#pragma unroll 1
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[16];
            tmem_ld16(tO + c * 16, o);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 16; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st16(tO + c * 16, o);
          }
        }
        if (r == 0) TRACE(t, 2, tr_it);
        const float neg_m = (m_used == -CUDART_INF_F) ? 0.f : -m_used;
        const float2 nm2 = make_float2(neg_m, neg_m);
        // P of one 16-column chunk, classified per warp: every row sees all of it (unmasked code),
        // no row sees any of it (zeros, no exponentials at all), or mixed - then all rows run the
        // masked code, which zeroes hidden columns after the exponential.  No divergence inside a
        // warp: per-row classes made a diagonal block three times as expensive as an interior one.
        auto exp16_body = [&](const float* v, int lim_k, uint32_t* pk, auto masked) {
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float2 x = fma2(make_float2(v[2 * i], v[2 * i + 1]), sc2, nm2);
            float2 e = (i & 3) < kEmuOf4 ? ex2_fma2(x) : make_float2(ex2(x.x), ex2(x.y));
            if (decltype(masked)::value) {
              if (2 * i > lim_k) e.x = 0.f;
              if (2 * i + 1 > lim_k) e.y = 0.f;
            }
            l2 = add2(l2, e);
            pk[i] = pack_bf16(e.x, e.y);
          }
        };
        auto exp16 = [&](const float* v, int k16, uint32_t* pk) {
          const int lim_k = lim - k16;
          if (!edge || lim_lo - k16 >= 15) {
            exp16_body(v, lim_k, pk, std::false_type{});
          } else if (lim_hi - k16 < 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) pk[i] = 0u;
          } else {
            exp16_body(v, lim_k, pk, std::true_type{});
          }
        };
#define RELOAD(addr, dst) tmem_ld16(addr, reinterpret_cast<uint32_t*>(dst))
        auto hand_over = [&](int slot) {  // this warp's chunk of P is in TMEM
          tmem_wait_st();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&p_full[4 * t + slot]);
        };
        // chunk order 3, 2, 0, 1 (slots 0..3 of the P handoff).  The store of a chunk is only
        // waited for after the arithmetic of the next one, so tcgen05.wait::st finds it complete.
        uint32_t pk[8];
        RELOAD(tS + 32, A);  // (not kept from pass 1: A would be live across the O rescale)
        exp16(B, 48, pk);
        tmem_st8(tS + 48, pk);
        tmem_wait_ld();
        RELOAD(tS, B);
        exp16(A, 32, pk);
        hand_over(0);
        tmem_st8(tS + 32, pk);
        tmem_wait_ld();
        RELOAD(tS + 16, A);
        exp16(B, 0, pk);
        hand_over(1);
        tmem_st8(tS, pk);
        tmem_wait_ld();
        exp16(A, 16, pk);
        hand_over(2);
        tmem_st8(tS + 16, pk);
        hand_over(3);
        };
        if (edge_block) softmax_block(std::true_type{}); else softmax_block(std::false_type{});
        if (r == 0) TRACE(t, 3 + hf, tr_it);
        ++tr_it;
        ++cnt;
      }
      // ------------------------------------ epilogue ------------------------------------
      // rows that saw no key: the emulated exp2 leaves ~2^-125 per masked score in l
      if (r == 0 && hf == 0) UTRACE(t, 2, un);
      const float l_half = m_used == -CUDART_INF_F ? 0.f : l2.x + l2.y;
      xch_l[hf * 128] = l_half;
      bar_sync(1 + t, 2 * kTile);
      const float l = l_half + xch_l[(hf ^ 1) * 128];
      mbar_wait(&o_full[t], o_ph);
      o_ph ^= 1;
      if (r == 0 && hf == 0) UTRACE(t, 3, un);
      tc_fence_after();
      const float inv_l = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[16];
        tmem_ld16(tO + c * 16, o);
        tmem_wait_ld();
        if (c == 0 && r == 0 && hf == 0) UTRACE(t, 6, un);
        if (valid) {
          uint4 pk[2];
#pragma unroll
          for (int v = 0; v < 2; ++v) {
            pk[v].x = pack_bf16(__uint_as_float(o[8 * v + 0]) * inv_l, __uint_as_float(o[8 * v + 1]) * inv_l);
            pk[v].y = pack_bf16(__uint_as_float(o[8 * v + 2]) * inv_l, __uint_as_float(o[8 * v + 3]) * inv_l);
            pk[v].z = pack_bf16(__uint_as_float(o[8 * v + 4]) * inv_l, __uint_as_float(o[8 * v + 5]) * inv_l);
            pk[v].w = pack_bf16(__uint_as_float(o[8 * v + 6]) * inv_l, __uint_as_float(o[8 * v + 7]) * inv_l);
          }
          // row-per-thread stores: one whole 32-byte sector per instruction where the layout
          // allows (two half-used sectors per 16 columns cost twice the LSU transactions)
          if (p.wide_stores) {
            stg256(reinterpret_cast<uint4*>(o_ptr) + c * 2, pk[0], pk[1]);
          } else {
            reinterpret_cast<uint4*>(o_ptr)[c * 2] = pk[0];
            reinterpret_cast<uint4*>(o_ptr)[c * 2 + 1] = pk[1];
          }
        }
      }
      if (r == 0 && hf == 0) UTRACE(t, 7, un);
      if (valid && hf == 0)
        p.LSE[(int64_t)h * p.lse_head_stride + grow] =
            l > 0.f ? m_used * 0.69314718055994531f + __logf(l) : -CUDART_INF_F;
      if (r == 0 && hf == 0) UTRACE(t, 4, un);
      if (r == 0 && hf == 0) UTRACE_VALUE(t, 5, un, tot);
      tc_fence_before();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kMmaWarp0) tmem_dealloc<512>(tmem);
}

}  // namespace

extern "C" {

bs_status_t bs_attn_workspace_bytes(const bs_attn_shape_t* shape, int32_t n_segs, int bwd,
                                    size_t* bytes) {
  bs_status_t rc = bs::validate_shape(shape, "bs_attn_workspace_bytes");
  if (rc != BS_OK) return rc;
  BS_REQUIRE(bytes != nullptr && n_segs >= 0, BS_ERR_INVALID_ARG,
             "bs_attn_workspace_bytes: bad arguments");
  *bytes = bs::ws_upper_bound(bwd ? shape->kv_rows : shape->q_rows, n_segs, bwd != 0);
  return BS_OK;
}

bs_status_t bs_attn_fwd(const bs_attn_shape_t* shape, const void* Q, const void* K, const void* V,
                        const bs_seg_t* segs, int32_t n_segs, int32_t out_row_begin,
                        int32_t out_row_end, void* O, float* LSE, void* ws, size_t ws_bytes,
                        void* stream, float* dQ_acc_clear) {
  bs_status_t rc = bs::validate_shape(shape, "bs_attn_fwd");
  if (rc != BS_OK) return rc;
  BS_REQUIRE(Q && K && V && O && LSE, BS_ERR_INVALID_ARG, "bs_attn_fwd: null tensor pointer");
  BS_REQUIRE(n_segs >= 0 && (segs || n_segs == 0), BS_ERR_INVALID_ARG, "bs_attn_fwd: bad segs");
  BS_REQUIRE(0 <= out_row_begin && out_row_begin <= out_row_end && out_row_end <= shape->q_rows,
             BS_ERR_INVALID_ARG, "bs_attn_fwd: output rows [%d,%d) outside [0,%d)", out_row_begin,
             out_row_end, shape->q_rows);
  BS_REQUIRE(((uintptr_t)O & 15) == 0, BS_ERR_INVALID_ARG, "bs_attn_fwd: O not 16-byte aligned");
  BS_REQUIRE(((uintptr_t)dQ_acc_clear & 15) == 0, BS_ERR_INVALID_ARG,
             "bs_attn_fwd: dQ_acc_clear not 16-byte aligned");
  if (out_row_end == out_row_begin) return BS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  // Everything that can fail on an argument comes first: work list, workspace, device, tensor
  // maps (pointer / stride alignment).  Nothing is enqueued before all of it has passed.
  bs::SchedTables tb;
  rc = bs::build_fwd_tables(segs, n_segs, shape->q_rows, shape->kv_rows, out_row_begin, out_row_end,
                            shape->n_q_heads, &tb);
  if (rc != BS_OK) return rc;
  bs::WsLayout L;
  rc = bs::check_workspace(tb, tb.clip_span_rows.size() * bs::kTensorMapBytes, ws, ws_bytes, &L);
  if (rc != BS_OK) return rc;
  rc = bs::check_device();
  if (rc != BS_OK) return rc;
  const int D = shape->head_dim;
  // V maps cut at every key range end that is not tile-aligned (TMA zero-fills past the end)
  rc = bs::append_clipped_maps(&tb, 0, 1, tb.clip_span_rows, V, D, shape->n_kv_heads,
                               shape->kv_row_stride);
  if (rc != BS_OK) return rc;
  CUtensorMap tmQ, tmK, tmV, tmZ;
  rc = bs::make_tensor_map_3d(&tmQ, Q, 2, D, shape->n_q_heads, shape->q_rows, shape->q_row_stride,
                              64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmK, K, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmV, V, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  // zero stores: rows clipped at out_row_end by the map itself (a unit's 256 rows may overhang)
  rc = bs::make_tensor_map_3d(&tmZ, dQ_acc_clear ? (const void*)dQ_acc_clear : Q, 4, D,
                              shape->n_q_heads, out_row_end, (int64_t)shape->n_q_heads * D, 32, 64, 0);
  if (rc != BS_OK) return rc;

  rc = bs::upload_tables(tb, L, ws, st);
  if (rc != BS_OK) return rc;
  uint8_t* wsb = (uint8_t*)ws;
  rc = bs::launch_fill_rows((const int2*)(wsb + L.fill_off), (int)tb.fill.size(), tb.max_fill_rows,
                            O, nullptr, LSE, shape->n_q_heads, shape->head_dim, shape->q_row_stride,
                            shape->lse_head_stride, st);
  if (rc != BS_OK) return rc;
  if (dQ_acc_clear != nullptr) {  // rows covered by no unit: cleared here (rare path)
    const size_t row_bytes = (size_t)shape->n_q_heads * D * sizeof(float);
    for (const bs::RowRange& f : tb.fill)
      BS_CUDA(cudaMemsetAsync((uint8_t*)dQ_acc_clear + (size_t)f.begin * row_bytes, 0,
                              (size_t)(f.end - f.begin) * row_bytes, st));
  }
  if (tb.items.empty()) return BS_OK;

  FwdParams p;
  p.clear_acc = dQ_acc_clear != nullptr;
  p.wide_stores = ((uintptr_t)O & 31) == 0 && (shape->q_row_stride * 2) % 32 == 0 && (D * 2) % 32 == 0;
  p.sv = bs::make_sched_view(wsb, L, tb, shape->n_q_heads);
  p.n_q_heads = shape->n_q_heads;
  p.group = shape->n_q_heads / shape->n_kv_heads;
  p.q_rows = shape->q_rows;
  const float scale = shape->softmax_scale > 0.f ? shape->softmax_scale : 1.f / sqrtf((float)D);
  p.scale_log2 = scale * 1.4426950408889634f;
  p.O = (__nv_bfloat16*)O;
  p.LSE = LSE;
  p.o_row_stride = shape->q_row_stride;
  p.lse_head_stride = shape->lse_head_stride;
  const int grid = tb.n_units < bs::sm_count() ? tb.n_units : bs::sm_count();
  if (D == 128) {
    rc = bs::set_max_smem_once((const void*)attn_fwd_kernel<128>, FwdSmem<128>::kAlloc, 0);
    if (rc != BS_OK) return rc;
    attn_fwd_kernel<128><<<grid, kFwdThreads, FwdSmem<128>::kAlloc, st>>>(tmQ, tmK, tmV, tmZ, p);
  } else {
    rc = bs::set_max_smem_once((const void*)attn_fwd_kernel<64>, FwdSmem<64>::kAlloc, 1);
    if (rc != BS_OK) return rc;
    attn_fwd_kernel<64><<<grid, kFwdThreads, FwdSmem<64>::kAlloc, st>>>(tmQ, tmK, tmV, tmZ, p);
  }
  BS_CUDA(cudaGetLastError());
  bs::count_launch();
  return BS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// bs_attn_fwd_static — the forward for callers that may not allocate (include/bytescale_attn.h).
// Same kernels and results as bs_attn_fwd; what differs is where the scratch lives (the array
// below instead of a caller workspace) and how the tables get there (kernel parameters of a copy
// kernel instead of a DMA from the library's pinned ring, which is allocated lazily).
// ------------------------------------------------------------------------------------------------
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

namespace {

constexpr size_t kStaticScratchBytes = BS_ATTN_STATIC_SCRATCH_BYTES;
// Held by every GPU that loads this library, until the process exits.  In HOST code this name is
// a host-side stand-in, not a device address: kernels get the address cudaGetSymbolAddress
// returns (static_scratch_address below), never `g_static_scratch` itself.
static __device__ __align__(256) uint8_t g_static_scratch[kStaticScratchBytes];

constexpr int kChunkBytes = 3584;  // per launch; the classic 4 KB parameter space minus the rest
struct TableChunk {
  uint4 v[kChunkBytes / 16];
};
static_assert(sizeof(TableChunk) == kChunkBytes && kChunkBytes % 256 == 0, "chunk size");

// dst[0 .. n_vec) = the chunk.  The tables include tensor maps, which the forward's TMA warp reads
// through the tensormap proxy after its own acquire fence; the release half goes here.
__global__ void __launch_bounds__(kChunkBytes / 16)
static_scratch_upload_kernel(const __grid_constant__ TableChunk c, uint4* dst, int n_vec) {
  const int i = threadIdx.x;
  if (i < n_vec) dst[i] = c.v[i];
  __threadfence();
  asm volatile("fence.proxy.tensormap::generic.release.gpu;" ::: "memory");
}

constexpr int kMaxScratchDevices = 64;
std::mutex g_scratch_mu;
uint8_t* g_scratch_addr[kMaxScratchDevices];  // device address of g_static_scratch, per device

// Set-up, once per device, with that device current.
bs_status_t static_scratch_address(uint8_t** out) {
  int dev = 0;
  BS_CUDA(cudaGetDevice(&dev));
  BS_REQUIRE(dev >= 0 && dev < kMaxScratchDevices, BS_ERR_UNSUPPORTED, "device index %d", dev);
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (g_scratch_addr[dev] == nullptr) {
    void* ptr = nullptr;
    BS_CUDA(cudaGetSymbolAddress(&ptr, g_static_scratch));
    BS_REQUIRE(ptr != nullptr && ((uintptr_t)ptr & 255) == 0, BS_ERR_CUDA,
               "bs_attn_fwd_static: scratch symbol address %p", ptr);
    g_scratch_addr[dev] = (uint8_t*)ptr;
  }
  *out = g_scratch_addr[dev];
  return BS_OK;
}

// [header | items | spans | groups | fill | tensor maps] as upload_tables (host_runtime.cpp) lays
// them out, into host memory.  Everything the kernels read is written, the cursor as 0.
void write_table_image(const bs::SchedTables& tb, const bs::WsLayout& L, uint8_t* img) {
  memset(img, 0, L.total);
  bs::SchedHeader* hd = reinterpret_cast<bs::SchedHeader*>(img);
  hd->counter = 0;
  hd->n_items = (int32_t)tb.items.size();
  hd->n_spans = (int32_t)tb.spans.size();
  hd->n_fill = (int32_t)tb.fill.size();
  hd->n_groups = (int32_t)tb.groups.size();
  hd->n_units = tb.n_units;
  if (!tb.groups.empty())
    memcpy(img + L.groups_off, tb.groups.data(), tb.groups.size() * sizeof(bs::Group));
  if (!tb.items.empty())
    memcpy(img + L.items_off, tb.items.data(), tb.items.size() * sizeof(bs::Item));
  if (!tb.spans.empty())
    memcpy(img + L.spans_off, tb.spans.data(), tb.spans.size() * sizeof(bs::Span));
  if (!tb.fill.empty())
    memcpy(img + L.fill_off, tb.fill.data(), tb.fill.size() * sizeof(bs::RowRange));
  if (!tb.tmaps.empty()) memcpy(img + L.tmaps_off, tb.tmaps.data(), tb.tmaps.size());
}

}  // namespace

extern "C" bs_status_t bs_attn_fwd_static(const bs_attn_shape_t* shape, const void* Q, const void* K,
                                          const void* V, const bs_seg_t* segs, int32_t n_segs,
                                          int32_t out_row_begin, int32_t out_row_end, void* O,
                                          float* LSE, void* stream, float* dQ_acc_clear) {
  bs_status_t rc = bs::validate_shape(shape, "bs_attn_fwd_static");
  if (rc != BS_OK) return rc;
  BS_REQUIRE(Q && K && V && O && LSE, BS_ERR_INVALID_ARG, "bs_attn_fwd_static: null tensor pointer");
  BS_REQUIRE(n_segs >= 0 && (segs || n_segs == 0), BS_ERR_INVALID_ARG,
             "bs_attn_fwd_static: bad segs");
  BS_REQUIRE(0 <= out_row_begin && out_row_begin <= out_row_end && out_row_end <= shape->q_rows,
             BS_ERR_INVALID_ARG, "bs_attn_fwd_static: output rows [%d,%d) outside [0,%d)",
             out_row_begin, out_row_end, shape->q_rows);
  BS_REQUIRE(((uintptr_t)O & 15) == 0, BS_ERR_INVALID_ARG,
             "bs_attn_fwd_static: O not 16-byte aligned");
  BS_REQUIRE(((uintptr_t)dQ_acc_clear & 15) == 0, BS_ERR_INVALID_ARG,
             "bs_attn_fwd_static: dQ_acc_clear not 16-byte aligned");
  if (out_row_end == out_row_begin) return BS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  // As in bs_attn_fwd, everything that can fail on an argument comes before the first enqueue.
  bs::SchedTables tb;
  rc = bs::build_fwd_tables(segs, n_segs, shape->q_rows, shape->kv_rows, out_row_begin, out_row_end,
                            shape->n_q_heads, &tb);
  if (rc != BS_OK) return rc;
  const bs::WsLayout L =
      bs::ws_layout(tb.items.size(), tb.spans.size(), tb.groups.size(), tb.fill.size(),
                    tb.clip_span_rows.size() * bs::kTensorMapBytes);
  BS_REQUIRE(L.total <= kStaticScratchBytes, BS_ERR_WORKSPACE,
             "bs_attn_fwd_static: the work list of this call needs %zu bytes of scratch, the "
             "library's static scratch holds %zu (BS_ATTN_STATIC_SCRATCH_BYTES); use bs_attn_fwd "
             "with a caller workspace",
             L.total, kStaticScratchBytes);
  rc = bs::check_device();
  if (rc != BS_OK) return rc;
  uint8_t* wsb = nullptr;
  rc = static_scratch_address(&wsb);
  if (rc != BS_OK) return rc;
  const int D = shape->head_dim;
  rc = bs::append_clipped_maps(&tb, 0, 1, tb.clip_span_rows, V, D, shape->n_kv_heads,
                               shape->kv_row_stride);
  if (rc != BS_OK) return rc;
  CUtensorMap tmQ, tmK, tmV, tmZ;
  rc = bs::make_tensor_map_3d(&tmQ, Q, 2, D, shape->n_q_heads, shape->q_rows, shape->q_row_stride,
                              64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmK, K, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmV, V, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmZ, dQ_acc_clear ? (const void*)dQ_acc_clear : Q, 4, D,
                              shape->n_q_heads, out_row_end, (int64_t)shape->n_q_heads * D, 32, 64, 0);
  if (rc != BS_OK) return rc;
  std::vector<uint8_t> img;  // host heap
  try {
    img.resize((L.total + kChunkBytes - 1) / kChunkBytes * kChunkBytes);
  } catch (const std::bad_alloc&) {
    return bs::fail(BS_ERR_HOST_OOM, "bs_attn_fwd_static: out of host memory (%zu bytes)", L.total);
  }
  write_table_image(tb, L, img.data());

  // Tables -> scratch, a chunk per launch, by value: the launch copies the chunk into the
  // parameter buffer, so `img` is dead when the loop ends.  Every byte the kernels below read
  // (the cursor at offset 0 included) is rewritten, whatever the previous call left.
  for (size_t off = 0; off < L.total; off += kChunkBytes) {
    const size_t n = L.total - off < (size_t)kChunkBytes ? L.total - off : (size_t)kChunkBytes;
    static_scratch_upload_kernel<<<1, kChunkBytes / 16, 0, st>>>(
        *reinterpret_cast<const TableChunk*>(img.data() + off),
        reinterpret_cast<uint4*>(wsb + off), (int)(n / 16));
    BS_CUDA(cudaGetLastError());
    bs::count_launch();
  }
  rc = bs::launch_fill_rows((const int2*)(wsb + L.fill_off), (int)tb.fill.size(), tb.max_fill_rows,
                            O, nullptr, LSE, shape->n_q_heads, shape->head_dim, shape->q_row_stride,
                            shape->lse_head_stride, st);
  if (rc != BS_OK) return rc;
  if (dQ_acc_clear != nullptr) {
    const size_t row_bytes = (size_t)shape->n_q_heads * D * sizeof(float);
    for (const bs::RowRange& f : tb.fill)
      BS_CUDA(cudaMemsetAsync((uint8_t*)dQ_acc_clear + (size_t)f.begin * row_bytes, 0,
                              (size_t)(f.end - f.begin) * row_bytes, st));
  }
  if (tb.items.empty()) return BS_OK;

  FwdParams p;
  p.clear_acc = dQ_acc_clear != nullptr;
  p.wide_stores = ((uintptr_t)O & 31) == 0 && (shape->q_row_stride * 2) % 32 == 0 && (D * 2) % 32 == 0;
  p.sv = bs::make_sched_view(wsb, L, tb, shape->n_q_heads);
  p.n_q_heads = shape->n_q_heads;
  p.group = shape->n_q_heads / shape->n_kv_heads;
  p.q_rows = shape->q_rows;
  const float scale = shape->softmax_scale > 0.f ? shape->softmax_scale : 1.f / sqrtf((float)D);
  p.scale_log2 = scale * 1.4426950408889634f;
  p.O = (__nv_bfloat16*)O;
  p.LSE = LSE;
  p.o_row_stride = shape->q_row_stride;
  p.lse_head_stride = shape->lse_head_stride;
  const int grid = tb.n_units < bs::sm_count() ? tb.n_units : bs::sm_count();
  if (D == 128) {
    rc = bs::set_max_smem_once((const void*)attn_fwd_kernel<128>, FwdSmem<128>::kAlloc, 0);
    if (rc != BS_OK) return rc;
    attn_fwd_kernel<128><<<grid, kFwdThreads, FwdSmem<128>::kAlloc, st>>>(tmQ, tmK, tmV, tmZ, p);
  } else {
    rc = bs::set_max_smem_once((const void*)attn_fwd_kernel<64>, FwdSmem<64>::kAlloc, 1);
    if (rc != BS_OK) return rc;
    attn_fwd_kernel<64><<<grid, kFwdThreads, FwdSmem<64>::kAlloc, st>>>(tmQ, tmK, tmV, tmZ, p);
  }
  BS_CUDA(cudaGetLastError());
  bs::count_launch();
  return BS_OK;
}
