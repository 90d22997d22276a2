// attn_bwd.cu — bs_attn_bwd: backward of one Q-chunk x KV-chunk step on sm_100a (SURVEY.md 8(a)
// a6; gradients of softmax attention as in flash-attention backward).
//
// One persistent CTA per SM, 512 threads, registers re-split by setmaxnreg (144 / 64 / 160):
//   warps 0-3   compute warpgroup A: query columns  0..63  of the transposed 128x128 tile
//   warps 4-7   compute warpgroup B: query columns 64..127
//   warp  8     MMA issuer (under elect_one: uniform-register descriptors, back-to-back UTCHMMA)
//   warp  9     TMA producer (+ LSE/delta staging)       warp 10  scheduler (sched.cuh)
//   warps 12-15 dQ drain warpgroup: TMEM -> registers -> shared -> TMA reduce-add into dQ_acc
// A unit is (one 128-key tile of a key range, one KV head).  The CTA keeps dK and dV of the tile
// in TMEM and loops over the G query heads of the group and over every 128-row query tile that
// sees the key tile; per iteration it issues the five MMAs of flash-attention backward, all with
// keys on the TMEM lanes ("transposed" form, thread r <-> key row r):
//   S^T  = K Q^T                  (SS)   -> P^T = exp2(S^T c - LSE)        written back to TMEM
//   dP^T = V dO^T                 (SS)   -> dS^T = P^T * (dP^T - delta) c  written to smem (bf16)
//   dV  += P^T dO                 (TS, A = P^T from TMEM, B = dO MN-major)
//   dQ   = dS K                   (SS, A = dS^T read MN-major, B = K MN-major)
//   dK  += dS^T Q                 (SS, A = dS^T K-major, B = Q MN-major)
// TMEM: X [0,128) S^T -> P^T in place -> S^T of the next iteration (behind dV in issue order);
//       Y [128,256) dP^T(n) -> dQ(n) -> dP^T(n+1): the drain warpgroup lifts dQ into registers the
//       moment it is complete, while dK(n) is still running;   [256,256+D) dK   [384,384+D) dV.
// Issue order per iteration n:  dP^T(n) | dV(n) S^T(n+1) | dQ(n) dK(n).  dP^T does not depend on P,
// so it runs under the compute warps' P step and dS follows P at once; the dependent chain is
// dS(n) -> dQ(n), dK(n), dP^T(n+1) -> dS(n+1).
// dK/dV are reduced over the group's heads inside the kernel (no atomics); dQ is reduced across
// key tiles and steps by the TMA unit in L2.  Measured: per iteration ~576 KB go
// through shared memory (MMA operands 288, dQ staging 128, dS 96, Q/dO loads 64) = ~4500 cycles at
// 128 B/clk against 2560 cycles of MMA math: this single-CTA SS-MMA form is shared-memory bound.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.h"
#include "launch_utils.h"
#include <type_traits>
#include "ptx.cuh"
#include "sched.cuh"
#include "worklist.h"

#define BS_TRACE_KERNEL_BWD
#include "trace.cuh"

namespace {

using namespace bs;
using namespace bs::ptx;

#ifndef BS_SCHED_SLOTS
#define BS_SCHED_SLOTS 1
#endif
constexpr int kBwdSchedSlots = BS_SCHED_SLOTS;  // depth of the scheduler ring (sched.cuh)
using SchedRing = SchedRingT<kBwdSchedSlots>;
using UnitProducer = UnitProducerT<kBwdSchedSlots>;
using UnitConsumer = UnitConsumerT<kBwdSchedSlots>;
constexpr int kSchedRingBytes = SchedRing::kBytes;

constexpr int kBwdThreads = 512;   // 2 compute WGs, auxiliary WG (MMA, TMA, scheduler), dQ drain WG
#ifndef BS_BWD_REGS_C
#define BS_BWD_REGS_C 144
#define BS_BWD_REGS_A 64
#define BS_BWD_REGS_D 160
#endif
// setmaxnreg split: compute, auxiliary, drain warpgroups: 2 c + a + d = 4 * 128
constexpr int kRegsCompute = BS_BWD_REGS_C, kRegsAux = BS_BWD_REGS_A, kRegsDrain = BS_BWD_REGS_D;
static_assert(2 * kRegsCompute + kRegsAux + kRegsDrain == 512, "register split");
constexpr int kComputeThreads = 256;
#ifndef BS_BWD_EMU
#define BS_BWD_EMU 0  // (1 of 4 was worth ~1 % before the dQ boxes became whole lines; now 0 is 2 % faster on cfg2)
#endif
constexpr int kBwdEmuOf4 = BS_BWD_EMU;  // of every 4 column pairs, this many take the FMA-pipe exp2

struct BwdParams {
  SchedView sv;     // units = key-tile items x n_kv_heads
  int32_t n_kv_heads, group;
  int32_t q_rows;
  float scale, scale_log2;
  const float* LSE;
  const float* delta;
  int64_t lse_head_stride;
  __nv_bfloat16* dK;
  __nv_bfloat16* dV;
  int64_t kv_row_stride;
  float* dQ_acc;  // [q_rows][Hq][D] fp32 dense
  int32_t n_q_heads;
};

template <int D>
struct BwdSmem {
  static constexpr int kTileBytes = kTile * D * 2;      // K, V, Q, dO tiles
  static constexpr int kKOff = 0;
  static constexpr int kVOff = kTileBytes;
  static constexpr int kQOff = 2 * kTileBytes;          // 2 stages
  static constexpr int kDOOff = 4 * kTileBytes;         // 1 stage
  static constexpr int kDSOff = 5 * kTileBytes;         // dS^T [128 keys][128 queries] bf16
  static constexpr int kDQOff = kDSOff + kTile * kTile * 2;  // 2 x [128][32] fp32 staging (dQ), 16 KB boxes
  static constexpr int kLseOff = kDQOff + 2 * kTile * 128;   // [2 stages][128] lse*log2e
  static constexpr int kDeltaOff = kLseOff + 2 * kTile * 4;  // [2 stages][128] delta*scale
  static constexpr int kBarOff = kDeltaOff + 2 * kTile * 4;
  // k_full k_empty (+ v_full v_empty at the end) q_full[2] q_empty[2] do_full do_empty s_full p_full dp_full ds_full dq_full
  // dq_drained acc_full acc_empty
  static constexpr int kNumBars = 19;
  static constexpr int kTmemSlotOff = kBarOff + kNumBars * 8;
  static constexpr int kSchedOff = kTmemSlotOff + 16;
  static constexpr int kBytes = kSchedOff + kSchedRingBytes;
};

// Iterations of one item: for each query head of the group, for each span (query range), the
// 128-row query tiles holding at least one query that sees the key tile's first key.
struct BwdWalker {
  const Span* table;
  const Unit* u;
  int n_spans, group, b0, hi, s, qi, n_qt;
  Span sp;
  __device__ __forceinline__ void load_span() {
    while (hi < group) {
      while (s < n_spans) {
        sp = unit_span(*u, table, s);
        const int a_min = max(0, b0 - sp.off);  // first query that sees key b0
        if (a_min < sp.len) {
          qi = a_min / kTile;
          n_qt = (sp.len + kTile - 1) / kTile;
          return;
        }
        ++s;
      }
      ++hi;
      s = 0;
    }
  }
  __device__ __forceinline__ void init(const Span* sp_table, const Unit& unit, int g) {
    const Item& it = unit.item;
    table = sp_table;
    u = &unit;
    n_spans = it.n_spans;
    group = g;
    b0 = it.local0;
    hi = 0;
    s = 0;
    load_span();
  }
  __device__ __forceinline__ bool done() const { return hi >= group; }
  __device__ __forceinline__ void next() {
    if (++qi >= n_qt) {
      ++s;
      load_span();
    }
  }
  __device__ __forceinline__ int q_row() const { return sp.begin + qi * kTile; }
};

// SS MMA, both operands K-major 128-row tiles (S^T = K Q^T, dP^T = V dO^T)
template <int D>
__device__ __forceinline__ void issue_kmajor(uint32_t tmem_d, uint32_t a_addr, uint32_t b_addr) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, kTile, 0, 0);
#pragma unroll
  for (int kk = 0; kk < D / 16; ++kk) {
    const uint32_t o = (kk / 4) * (kTile * 128) + (kk % 4) * 32;
    umma_ss(tmem_d, umma_desc_sw128(a_addr + o, 16, 1024), umma_desc_sw128(b_addr + o, 16, 1024),
            idesc, kk > 0);
  }
}
// dV += P^T dO : A from TMEM (packed bf16), B = dO [queries][D] MN-major
template <int D>
__device__ __forceinline__ void issue_dv(uint32_t tmem_d, uint32_t tmem_p, uint32_t do_addr,
                                         bool accumulate) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, D, 0, 1);
#pragma unroll
  for (int kk = 0; kk < kTile / 16; ++kk)
    umma_ts(tmem_d, tmem_p + (kk / 4) * 64 + (kk % 4) * 8,  // P^T halves at columns [0,32), [64,96)
            umma_desc_sw128(do_addr + kk * 2048, kTile * 128, 1024), idesc, accumulate || kk > 0);
}
// dK += dS^T Q : A = dS^T [keys][queries] K-major (two 64-query boxes), B = Q MN-major
template <int D>
__device__ __forceinline__ void issue_dk(uint32_t tmem_d, uint32_t ds_addr, uint32_t q_addr,
                                         bool accumulate) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, D, 0, 1);
#pragma unroll
  for (int kk = 0; kk < kTile / 16; ++kk) {
    const uint32_t o = (kk / 4) * (kTile * 128) + (kk % 4) * 32;
    umma_ss(tmem_d, umma_desc_sw128(ds_addr + o, 16, 1024),
            umma_desc_sw128(q_addr + kk * 2048, kTile * 128, 1024), idesc, accumulate || kk > 0);
  }
}
// dQ = dS K : A = the same dS^T smem read MN-major (M = queries contiguous), B = K MN-major
template <int D>
__device__ __forceinline__ void issue_dq(uint32_t tmem_d, uint32_t ds_addr, uint32_t k_addr) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, D, 1, 1);
#pragma unroll
  for (int kk = 0; kk < kTile / 16; ++kk)
    umma_ss(tmem_d, umma_desc_sw128(ds_addr + kk * 2048, kTile * 128, 1024),
            umma_desc_sw128(k_addr + kk * 2048, kTile * 128, 1024), idesc, kk > 0);
}

}  // namespace

namespace {

// all lanes of a converged warp have finished their part: one arrival for the warp
__device__ __forceinline__ void warp_arrive(uint64_t* bar) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(bar);
}

template <int D>
__global__ void __launch_bounds__(kBwdThreads, 1)
attn_bwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmDO,
                const __grid_constant__ CUtensorMap tmDQ, const __grid_constant__ CUtensorMap tmDK,
                const __grid_constant__ CUtensorMap tmDV, const __grid_constant__ BwdParams p) {
  using L = BwdSmem<D>;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::kBarOff);
  uint64_t* k_full = bars + 0;
  uint64_t* k_empty = bars + 1;
  uint64_t* v_full = bars + 16;
  uint64_t* v_empty = bars + 17;
  uint64_t* q_full = bars + 2;   // [2]
  uint64_t* q_empty = bars + 4;  // [2]
  uint64_t* do_full = bars + 6;
  uint64_t* do_empty = bars + 7;
  uint64_t* s_full = bars + 8;
  uint64_t* p_full = bars + 9;
  uint64_t* dp_full = bars + 10;
  uint64_t* ds_full = bars + 11;
  uint64_t* dq_full = bars + 12;
  uint64_t* dq_drained = bars + 13;
  uint64_t* acc_full = bars + 14;
  uint64_t* acc_empty = bars + 15;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kTmemSlotOff);
  float* lse_s = reinterpret_cast<float*>(smem + L::kLseOff);
  float* delta_s = reinterpret_cast<float*>(smem + L::kDeltaOff);
  SchedRing* sched = reinterpret_cast<SchedRing*>(smem + L::kSchedOff);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0 && (smem_u32(smem) & 1023u) != 0) {
    printf("bs_attn_bwd: dynamic shared memory base is not 1024-byte aligned\n");
    __trap();
  }
  if (warp == 9 && lane == 0) {
    // arrivals per unit: one per compute warp, the MMA lane, the TMA lane, one per drain warp
    sched_ring_init(sched, kComputeThreads / 32 + 2 + kTile / 32);
    mbar_init(k_full, 1);
    mbar_init(k_empty, 1);
    mbar_init(v_full, 1);
    mbar_init(v_empty, 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&q_full[i], 33);  // expect_tx arrive + 32 lanes staging LSE/delta
      mbar_init(&q_empty[i], 1);
    }
    mbar_init(do_full, 1);
    mbar_init(do_empty, 1);
    mbar_init(s_full, 1);
    mbar_init(p_full, kComputeThreads / 32);  // one arrival per compute warp
    mbar_init(dp_full, 1);
    mbar_init(ds_full, kComputeThreads / 32);  // one arrival per compute warp
    mbar_init(dq_full, 1);
    mbar_init(dq_drained, 4);  // one arrival per drain warp
    mbar_init(acc_full, 1);
    mbar_init(acc_empty, kComputeThreads / 32);  // one arrival per compute warp
    fence_barrier_init();
    prefetch_tensormap(&tmQ);
    prefetch_tensormap(&tmK);
    prefetch_tensormap(&tmV);
    prefetch_tensormap(&tmDO);
    prefetch_tensormap(&tmDQ);
    prefetch_tensormap(&tmDK);
    prefetch_tensormap(&tmDV);
  }
  if (warp == 8) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t sK = smem_u32(smem + L::kKOff), sV = smem_u32(smem + L::kVOff);
  const uint32_t sQ = smem_u32(smem + L::kQOff), sDO = smem_u32(smem + L::kDOOff);
  const uint32_t sDS = smem_u32(smem + L::kDSOff);

  if (warp >= 8 && warp < 12) setmaxnreg_dec<kRegsAux>();
  if (warp == 9) {
    // ============================ TMA producer + LSE/delta staging ============================
    // Ragged tiles - the last key tile of a key range, the last query tile of a query range -
    // are loaded through tensor maps whose row extent ends at the range end (host-built, in the
    // workspace): TMA zero-fills the rows past it.  A whole 128-row box through the buffer-wide
    // map would bring in whatever follows in the caller's buffer - another document, or
    // uninitialised rows with NaN / Inf - and 0 (masked P, dS) x NaN inside an MMA's contraction
    // would poison every output row of the tile.
    // A tensor map in global memory must be fenced by the thread that uses it (the workspace
    // address held other maps in earlier launches).  A fence costs ~360 cycles and the loads of
    // ragged tiles sit on the iteration's critical path (single-buffered dO), so every clipped
    // map is OWNED by one lane of this warp - lane 1 + index % 31 - which fences it once, up
    // front, and issues every load that goes through it; lane 0 issues all other loads.
    uint32_t item_n = 0, it_n = 0;  // items / iterations issued so far (ring phases)
    const CUtensorMap* clips_q = p.sv.tmaps;                           // [2 i] Q, [2 i + 1] dO
    const CUtensorMap* clips_k = p.sv.tmaps + 2 * p.sv.n_span_clips;   // [2 j] K, [2 j + 1] V
    if (lane > 0) {
      for (int c = lane - 1; c < p.sv.n_span_clips + p.sv.n_item_clips; c += 31) {
        tensormap_acquire(clips_q + 2 * c);
        tensormap_acquire(clips_q + 2 * c + 1);
      }
    }
    UnitConsumer cons{sched};  // lane 0 consumes; the other lanes read the slot after it
    while (true) {
      Unit u;
      if (lane != 0) cons.wait_peek(&u);
      __syncwarp();  // lane 0 releases the slot only after everybody has read it
      int more = 0;
      if (lane == 0) more = cons.next(&u);
      more = __shfl_sync(0xffffffffu, more, 0);
      if (lane != 0) ++cons.n;
      if (!more) break;
      const Item& it = u.item;
      const int g = u.head;
      BwdWalker wk;
      wk.init(p.sv.spans, u, p.group);
      if (wk.done()) continue;
      // The first iteration's Q / LSE / delta / dO go out BEFORE this unit's K and V: their
      // buffers free up well before the previous unit ends, whereas V is only released at that
      // unit's last dP^T MMA and K at its last dQ MMA.  K/V then stream in under the previous
      // unit's tail (dS, dK/dQ, the dQ drain and the dK/dV epilogue).
      const int kclip = it.tile_blocks[0];  // bwd: clipped K / V maps of this key tile, or -1
      const CUtensorMap* mK = kclip >= 0 ? clips_k + 2 * kclip : &tmK;
      const CUtensorMap* mV = kclip >= 0 ? mK + 1 : &tmV;
      const int own_k = kclip >= 0 ? 1 + (p.sv.n_span_clips + kclip) % 31 : 0;
      auto load_kv = [&]() {
        TRACE(2, 8, it_n);  // the producer is ready to load this unit's K / V
        mbar_wait(v_empty, (item_n & 1) ^ 1);
        mbar_arrive_expect_tx(v_full, L::kTileBytes);
        for (int half = 0; half < D / 64; ++half)
          tma_load_3d(smem + L::kVOff + half * (kTile * 128), mV, v_full, half * 64, g, it.row0);
        mbar_wait(k_empty, (item_n & 1) ^ 1);
        TRACE(2, 9, it_n);  // K requested
        mbar_arrive_expect_tx(k_full, L::kTileBytes);
        for (int half = 0; half < D / 64; ++half)
          tma_load_3d(smem + L::kKOff + half * (kTile * 128), mK, k_full, half * 64, g, it.row0);
      };
      bool kv_pending = true;
      for (; !wk.done(); wk.next(), ++it_n) {
        const int st = it_n & 1, h = g * p.group + wk.hi, qrow = wk.q_row();
        const bool qclip = wk.sp.clip >= 0 && wk.sp.len - wk.qi * kTile < kTile;
        const CUtensorMap* mQ = qclip ? clips_q + 2 * wk.sp.clip : &tmQ;
        const CUtensorMap* mDO = qclip ? mQ + 1 : &tmDO;
        const int own_q = qclip ? 1 + wk.sp.clip % 31 : 0;
        // -lse*log2e (-inf for rows outside the query range) and -delta*scale: fetched BEFORE the
        // wait for the stage (the producer runs ahead and sits in that wait), so that the ~800
        // cycles of L2 latency are not in front of this iteration's dO request
        float lse_v[kTile / 32], delta_v[kTile / 32];
#pragma unroll
        for (int k = 0; k < kTile / 32; ++k) {
          const int c = lane + 32 * k;
          const bool ok = wk.qi * kTile + c < wk.sp.len;
          const int64_t idx = (int64_t)h * p.lse_head_stride + qrow + c;
          // negated, so that the compute warps fold them in with one packed FMA each
          lse_v[k] = ok ? -__ldg(p.LSE + idx) * 1.4426950408889634f : -CUDART_INF_F;
          delta_v[k] = ok ? -__ldg(p.delta + idx) * p.scale : 0.f;
        }
        mbar_wait(&q_empty[st], ((it_n >> 1) & 1) ^ 1);
        if (lane == own_q) {
          mbar_arrive_expect_tx(&q_full[st], L::kTileBytes);
          for (int half = 0; half < D / 64; ++half)
            tma_load_3d(smem + L::kQOff + st * L::kTileBytes + half * (kTile * 128), mQ,
                        &q_full[st], half * 64, h, qrow);
        }
#pragma unroll
        for (int k = 0; k < kTile / 32; ++k) {
          lse_s[st * kTile + lane + 32 * k] = lse_v[k];
          delta_s[st * kTile + lane + 32 * k] = delta_v[k];
        }
        mbar_arrive(&q_full[st]);
        if (lane == own_q) {
          mbar_wait(do_empty, (it_n & 1) ^ 1);
          mbar_arrive_expect_tx(do_full, L::kTileBytes);
          for (int half = 0; half < D / 64; ++half)
            tma_load_3d(smem + L::kDOOff + half * (kTile * 128), mDO, do_full, half * 64, h, qrow);
        }
        if (kv_pending) {
          __syncwarp();  // K / V go out behind the first dO, whichever lanes issue them
          if (lane == own_k) load_kv();
        }
        kv_pending = false;
        __syncwarp();
      }
      ++item_n;
    }
  } else if (warp == 10) {
    // ======================================== scheduler ========================================
    if (lane == 0) {
      UnitProducer prod{sched};
      Unit u;
      while (prod.next(p.sv, &u)) {
      }
    }
  } else if (warp == 8) {
    // ======================================= MMA issuer =======================================
    // (elect_one, not lane == 0: the compiler then knows a single thread runs the region and
    // keeps the MMA descriptors in uniform registers - back-to-back UTCHMMA instead of a
    // broadcast loop of ~16 instructions per MMA, which made the issue itself the bottleneck)
    if (elect_one()) {
      uint32_t item_n = 0, it_n = 0;
      UnitConsumer cons{sched};
      Unit u;
      while (cons.next(&u)) {
        const Item& it = u.item;
        BwdWalker wk;
        wk.init(p.sv.spans, u, p.group);
        if (wk.done()) continue;
        TRACE(2, 5, it_n);  // unit picked up
        mbar_wait(k_full, item_n & 1);
        TRACE(2, 6, it_n);
        tc_fence_after();
        // prologue: S^T(0)
        mbar_wait(&q_full[it_n & 1], (it_n >> 1) & 1);
        TRACE(2, 7, it_n);
        tc_fence_after();
        issue_kmajor<D>(tmem, sK, sQ + (it_n & 1) * L::kTileBytes);
        tc_commit(s_full);
        bool first = true;
        while (true) {
          BwdWalker nxt = wk;
          nxt.next();
          const bool has_next = !nxt.done();
          const uint32_t st = it_n & 1;
          // dP^T = V dO^T first: it does not depend on P, so it runs under the compute warps' P
          // step and dS can follow P at once.  Its region held dQ of the previous iteration,
          // which the drain warpgroup lifts into registers as soon as it is complete.
          mbar_wait(do_full, it_n & 1);
          if (first) mbar_wait(v_full, item_n & 1);
          if (it_n > 0) mbar_wait(dq_drained, (it_n - 1) & 1);
          tc_fence_after();
          issue_kmajor<D>(tmem + 128, sV, sDO);
          tc_commit(dp_full);
          TRACE(2, 1, it_n);
          if (!has_next) tc_commit(v_empty);
          // dV += P^T dO
          mbar_wait(p_full, it_n & 1);
          if (first) mbar_wait(acc_empty, (item_n & 1) ^ 1);  // previous unit's dK/dV have left TMEM
          tc_fence_after();
          TRACE(2, 0, it_n);
          issue_dv<D>(tmem + 384, tmem, sDO, !first);
          tc_commit(do_empty);
          // S^T of the next iteration (P^T of this one has been consumed by dV, in issue order)
          if (has_next) {
            mbar_wait(&q_full[(it_n + 1) & 1], ((it_n + 1) >> 1) & 1);
            tc_fence_after();
            issue_kmajor<D>(tmem, sK, sQ + ((it_n + 1) & 1) * L::kTileBytes);
            tc_commit(s_full);
          }
          // dK += dS^T Q ; dQ = dS K (into the region dP^T was read from)
          TRACE(2, 2, it_n);
          mbar_wait(ds_full, it_n & 1);
          TRACE(2, 3, it_n);
          tc_fence_after();
          // dQ before dK: the next iteration's dP^T needs dQ's region back (the drain warpgroup
          // lifts dQ out while dK runs), and K is released one MMA group earlier at the unit's end
          issue_dq<D>(tmem + 128, sDS, sK);
          tc_commit(dq_full);
          if (!has_next) tc_commit(k_empty);
          issue_dk<D>(tmem + 256, sDS, sQ + st * L::kTileBytes, !first);
          tc_commit(&q_empty[st]);
          TRACE(2, 4, it_n);
          first = false;
          ++it_n;
          if (!has_next) break;
          wk = nxt;
        }
        tc_commit(acc_full);
        ++item_n;
      }
    }
  } else if (warp >= 12) {
    // ===================================== dQ drain warpgroup =====================================
    // dQ of every iteration: TMEM -> registers -> shared -> TMA reduce-add (fp32 add in L2) into
    // dQ_acc, 32 columns (one 16 KB box of 128 rows x 128 B, 128-byte swizzle) at a time through
    // two staging boxes: whole 128-byte lines per row on the way to L2 (with four 8 KB boxes of
    // 64-byte row segments the backward was 2-3 % slower - the SM's request path to L2 is 64 %
    // busy in this kernel, ncu l1tex__m_l1tex2xbar_req_cycles_active).  The TMA unit needs well
    // over 1000 cycles to read a box; that used to sit on the compute warps' critical path.  Only
    // the TMEM -> register lift is urgent (see the issuer).
    setmaxnreg_inc<kRegsDrain>();
    const int r = threadIdx.x & 127;  // query row of the tile
    const uint32_t tY = tmem + (uint32_t((warp & 3) * 32) << 16) + 128;
    uint8_t* stage0 = smem + L::kDQOff;
    uint32_t it_n = 0;
    UnitConsumer cons{sched};
    Unit u;
    while (cons.next_arrive_once(&u)) {
      const int g = u.head;
      BwdWalker wk;
      wk.init(p.sv.spans, u, p.group);
      for (; !wk.done(); wk.next(), ++it_n) {
        const int h = g * p.group + wk.hi, qrow = wk.q_row();
        mbar_wait(dq_full, it_n & 1);
        tc_fence_after();
        // all D columns into registers first: the region goes straight back to the MMA issuer,
        // whose next dP^T (on the critical path of the next iteration) is waiting for it
        uint32_t v[D];
#pragma unroll
        for (int c = 0; c < D / 32; ++c) tmem_ld32(tY + c * 32, &v[c * 32]);
        tmem_wait_ld();
        tc_fence_before();
        warp_arrive(dq_drained);
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint8_t* stage = stage0 + (c & 1) * 16384;
          if (r == 0) bulk_wait_group_read<1>();  // the reduce two chunks back has read this box
          bar_sync(3, 128);
#pragma unroll
          for (int j = 0; j < 8; ++j)
            *reinterpret_cast<uint4*>(stage + r * 128 + ((j ^ (r & 7)) * 16)) =
                make_uint4(v[32 * c + 4 * j], v[32 * c + 4 * j + 1], v[32 * c + 4 * j + 2],
                           v[32 * c + 4 * j + 3]);
          fence_proxy_async_smem();
          bar_sync(3, 128);
          if (r == 0) {
            tma_reduce_add_3d(&tmDQ, stage, c * 32, h, qrow);
            bulk_commit_group();
          }
        }
      }
    }
    if (r == 0) bulk_wait_group<0>();  // all dQ reductions have landed before the CTA exits
  } else if (warp < 8) {
    // ==================================== compute warpgroups ====================================
    setmaxnreg_inc<kRegsCompute>();
    const int wg = warp >> 2;
    const int r = threadIdx.x & 127;  // key row of the tile
    const uint32_t lane_addr = uint32_t((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + lane_addr + wg * 64;         // this half's S^T columns (fp32)
    const uint32_t tP = tS;                                  // its P^T (packed bf16), 32 columns
    const uint32_t tDP = tmem + lane_addr + 128 + wg * 64;  // this half's dP^T columns (region Y)
    uint8_t* ds_row = smem + L::kDSOff + wg * (kTile * 128) + r * 128;
    uint32_t item_n = 0, it_n = 0;
    UnitConsumer cons{sched};
    Unit u;
    while (cons.next_arrive_once(&u)) {
      const Item& it = u.item;
      const int g = u.head;
      const int b = it.local0 + r;  // key index inside its range
      const bool key_ok = b < it.range_len;
      BwdWalker wk;
      wk.init(p.sv.spans, u, p.group);
      __nv_bfloat16* out = (wg == 0 ? p.dK : p.dV) + ((int64_t)it.row0 + r) * p.kv_row_stride +
                           (int64_t)g * D;
      if (wk.done()) {  // no query sees this key tile: its gradients are zero
        if (key_ok)
          for (int c = 0; c < D / 8; ++c) reinterpret_cast<uint4*>(out)[c] = make_uint4(0, 0, 0, 0);
        continue;
      }
      uint32_t pk[32];  // P^T of this thread as the tensor core sees it (bf16 pairs), kept for dS
      bool first = true;

      auto compute_p = [&](const BwdWalker& k, uint32_t n) {
        mbar_wait(s_full, n & 1);
        if (r == 0) TRACE(wg, 0, n);
        tc_fence_after();
        uint32_t s[64];
        tmem_ld32(tS, &s[0]);
        tmem_ld32(tS + 32, &s[32]);
        tmem_wait_ld();
        const float2* nl2 = reinterpret_cast<const float2*>(lse_s + (n & 1) * kTile + wg * 64);
        const int a0 = k.qi * kTile + wg * 64;  // query index of this half's first column
        // column cc is visible iff c_min <= cc < c_max (key b <= query a0 + cc + off, query inside
        // its range); `full`: nothing of this warpgroup's 128 x 64 piece is masked (warp-uniform)
        const bool full = it.local0 + kTile - 1 <= a0 + k.sp.off && it.local0 + kTile <= it.range_len &&
                          a0 + 64 <= k.sp.len;
        const int c_min = key_ok ? b - k.sp.off - a0 : (1 << 30);
        const int c_max = k.sp.len - a0;
        const float2 sc2 = make_float2(p.scale_log2, p.scale_log2);
        // two copies of the loop: unmasked pieces (nearly all of them) run branch- and
        // predicate-free straight-line code
        auto exp_all = [&](auto masked) {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float2 x = fma2(make_float2(__uint_as_float(s[2 * i]), __uint_as_float(s[2 * i + 1])),
                                  sc2, nl2[i]);
            float2 e = (i & 3) < kBwdEmuOf4 ? ex2_fma2(x) : make_float2(ex2(x.x), ex2(x.y));
            if (decltype(masked)::value) {  // masked P exactly 0, whichever exp2 path produced it
              if (2 * i < c_min || 2 * i >= c_max) e.x = 0.f;
              if (2 * i + 1 < c_min || 2 * i + 1 >= c_max) e.y = 0.f;
            }
            pk[i] = pack_bf16(e.x, e.y);
          }
        };
        if (full) exp_all(std::false_type{}); else exp_all(std::true_type{});
        tmem_st32(tP, pk);
        tmem_wait_st();
        tc_fence_before();
        warp_arrive(p_full);
        if (r == 0) TRACE(wg, 1, n);
      };

      uint8_t* ds_box = smem + L::kDSOff + wg * (kTile * 128);

      while (true) {
        compute_p(wk, it_n);
        BwdWalker nxt = wk;
        nxt.next();
        const bool has_next = !nxt.done();
        // dS^T = P^T * (dP^T * scale - delta * scale)
        mbar_wait(dp_full, it_n & 1);
        if (r == 0) TRACE(wg, 2, it_n);
        tc_fence_after();
        {
          uint32_t dp[64];
          tmem_ld32(tDP, &dp[0]);
          tmem_ld32(tDP + 32, &dp[32]);
          tmem_wait_ld();
          if (r == 0) TRACE(wg, 8, it_n);
          if (first) {  // the previous unit's last dQ reduce / epilogue stores read this dS^T box
            if (r == 0) bulk_wait_group_read<0>();
            bar_sync(1 + wg, 128);
          }
          const float2* nd2 = reinterpret_cast<const float2*>(delta_s + (it_n & 1) * kTile + wg * 64);
          const float2 s2 = make_float2(p.scale, p.scale);
#pragma unroll
          for (int j = 0; j < 8; ++j) {  // 8 queries = one 16-byte chunk of the dS^T row
            uint32_t w4[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int i = 4 * j + e;
              const float2 t = fma2(make_float2(__uint_as_float(dp[2 * i]), __uint_as_float(dp[2 * i + 1])),
                                    s2, nd2[i]);
              // P widened exactly from the bf16 pair the dV MMA used.  Masked P is exactly 0 and
              // t is finite everywhere (rows past a range end are zero-filled by TMA, see the
              // producer), so masked dS is exactly 0 without a select.
              const float2 d = mul2(make_float2(__uint_as_float(pk[i] << 16),
                                                __uint_as_float(pk[i] & 0xffff0000u)), t);
              w4[e] = pack_bf16(d.x, d.y);
            }
            *reinterpret_cast<uint4*>(ds_row + ((j ^ (r & 7)) * 16)) = make_uint4(w4[0], w4[1], w4[2], w4[3]);
          }
        }
        if (r == 0) TRACE(wg, 9, it_n);
        fence_proxy_async_smem();
        tc_fence_before();
        warp_arrive(ds_full);
        if (r == 0) TRACE(wg, 3, it_n);
        first = false;
        ++it_n;
        if (!has_next) break;
        wk = nxt;
      }
      // ------------------------------ epilogue: dK (WG A), dV (WG B) ------------------------------
      if (r == 0) TRACE(wg, 5, it_n - 1);
      mbar_wait(acc_full, item_n & 1);
      if (r == 0) TRACE(wg, 6, it_n - 1);
      tc_fence_after();
      const uint32_t tAcc = tmem + lane_addr + 256 + wg * 128;
      if (it.local0 + kTile <= it.range_len) {
        // Full key tile: 32 columns at a time through this warpgroup's half of the dQ staging
        // area (two 8 KB buffers) and out with TMA stores - whole 64-byte row segments, no LSU
        // work.  (Row-per-thread 16-byte global stores cost one half-used sector each: ~5000
        // cycles per unit, measured.)
        // staging: the two 8 KB halves of this warpgroup's dS^T box (free: the unit's last dK / dQ
        // MMAs are complete)
        constexpr int kChunks = D / 32;
#pragma unroll
        for (int c = 0; c < kChunks; ++c) {
          uint32_t v[32];
          tmem_ld32(tAcc + c * 32, v);
          tmem_wait_ld();
          if (c == kChunks - 1) {  // the accumulators have left TMEM
            tc_fence_before();
            warp_arrive(acc_empty);
          }
          uint8_t* stg = ds_box + (c & 1) * 8192;
          if (r == 0) bulk_wait_group_read<1>();  // the store two chunks back has read this buffer
          bar_sync(1 + wg, 128);
          uint8_t* row = stg + r * 64;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint4 pk;
            pk.x = pack_bf16(__uint_as_float(v[8 * q + 0]), __uint_as_float(v[8 * q + 1]));
            pk.y = pack_bf16(__uint_as_float(v[8 * q + 2]), __uint_as_float(v[8 * q + 3]));
            pk.z = pack_bf16(__uint_as_float(v[8 * q + 4]), __uint_as_float(v[8 * q + 5]));
            pk.w = pack_bf16(__uint_as_float(v[8 * q + 6]), __uint_as_float(v[8 * q + 7]));
            *reinterpret_cast<uint4*>(row + ((q ^ ((r >> 1) & 3)) * 16)) = pk;  // 64-byte swizzle
          }
          fence_proxy_async_smem();
          bar_sync(1 + wg, 128);
          if (r == 0) {
            tma_store_3d(wg == 0 ? &tmDK : &tmDV, stg, c * 32, g, it.row0);
            bulk_commit_group();
          }
        }
      } else {
        // ragged last tile of a key range: rows past the range belong to somebody else
#pragma unroll
        for (int c = 0; c < D / 32; ++c) {
          uint32_t v[32];
          tmem_ld32(tAcc + c * 32, v);
          tmem_wait_ld();
          if (key_ok) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              uint4 pk;
              pk.x = pack_bf16(__uint_as_float(v[8 * q + 0]), __uint_as_float(v[8 * q + 1]));
              pk.y = pack_bf16(__uint_as_float(v[8 * q + 2]), __uint_as_float(v[8 * q + 3]));
              pk.z = pack_bf16(__uint_as_float(v[8 * q + 4]), __uint_as_float(v[8 * q + 5]));
              pk.w = pack_bf16(__uint_as_float(v[8 * q + 6]), __uint_as_float(v[8 * q + 7]));
              reinterpret_cast<uint4*>(out)[c * 4 + q] = pk;
            }
          }
        }
        tc_fence_before();
        warp_arrive(acc_empty);
      }
      if (r == 0) TRACE(wg, 7, it_n - 1);
      ++item_n;
    }
    if (r == 0) bulk_wait_group<0>();  // all dQ reductions have landed before the CTA exits
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc<512>(tmem);
}

}  // namespace

extern "C" bs_status_t bs_attn_bwd(const bs_attn_shape_t* shape, const void* Q, const void* K,
                                   const void* V, const void* dO, const float* LSE_final,
                                   const float* delta, const bs_seg_t* segs, int32_t n_segs,
                                   float* dQ_acc, void* dK, void* dV, void* ws, size_t ws_bytes,
                                   void* stream) {
  bs_status_t rc = bs::validate_shape(shape, "bs_attn_bwd");
  if (rc != BS_OK) return rc;
  BS_REQUIRE(Q && K && V && dO && LSE_final && delta && dQ_acc && dK && dV, BS_ERR_INVALID_ARG,
             "bs_attn_bwd: null tensor pointer");
  BS_REQUIRE(n_segs >= 0 && (segs || n_segs == 0), BS_ERR_INVALID_ARG, "bs_attn_bwd: bad segs");
  BS_REQUIRE((((uintptr_t)dK | (uintptr_t)dV | (uintptr_t)dQ_acc) & 15) == 0, BS_ERR_INVALID_ARG,
             "bs_attn_bwd: output pointers must be 16-byte aligned");
  if (shape->kv_rows == 0) return BS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  // Everything that can fail on an argument comes first: work list, workspace, device, tensor
  // maps (pointer / stride alignment).  Nothing is enqueued before all of it has passed.
  bs::SchedTables tb;
  rc = bs::build_bwd_tables(segs, n_segs, shape->q_rows, shape->kv_rows, shape->n_kv_heads, &tb);
  if (rc != BS_OK) return rc;
  bs::WsLayout L;
  const size_t n_qc = tb.clip_span_rows.size(), n_kc = tb.clip_item_rows.size();
  rc = bs::check_workspace(tb, 2 * (n_qc + n_kc) * bs::kTensorMapBytes, ws, ws_bytes, &L);
  if (rc != BS_OK) return rc;
  rc = bs::check_device();
  if (rc != BS_OK) return rc;
  const int D = shape->head_dim;
  // Q / dO maps cut at every query range end and K / V maps cut at every key range end that is
  // not tile-aligned (TMA zero-fills past the end): [2 i] Q, [2 i + 1] dO, then [2 j] K, [2 j + 1] V
  rc = bs::append_clipped_maps(&tb, 0, 2, tb.clip_span_rows, Q, D, shape->n_q_heads, shape->q_row_stride);
  if (rc == BS_OK)
    rc = bs::append_clipped_maps(&tb, 1, 2, tb.clip_span_rows, dO, D, shape->n_q_heads, shape->q_row_stride);
  if (rc == BS_OK)
    rc = bs::append_clipped_maps(&tb, 2 * n_qc, 2, tb.clip_item_rows, K, D, shape->n_kv_heads,
                                 shape->kv_row_stride);
  if (rc == BS_OK)
    rc = bs::append_clipped_maps(&tb, 2 * n_qc + 1, 2, tb.clip_item_rows, V, D, shape->n_kv_heads,
                                 shape->kv_row_stride);
  if (rc != BS_OK) return rc;
  CUtensorMap tmQ, tmK, tmV, tmDO, tmDQ, tmDK, tmDV;
  rc = bs::make_tensor_map_3d(&tmQ, Q, 2, D, shape->n_q_heads, shape->q_rows, shape->q_row_stride,
                              64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmDO, dO, 2, D, shape->n_q_heads, shape->q_rows,
                              shape->q_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmK, K, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmV, V, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmDQ, dQ_acc, 4, D, shape->n_q_heads, shape->q_rows,
                              (int64_t)shape->n_q_heads * D, 32, bs::kTile, 128);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmDK, dK, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 32, bs::kTile, 64);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmDV, dV, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 32, bs::kTile, 64);
  if (rc != BS_OK) return rc;

  rc = bs::upload_tables(tb, L, ws, st);
  if (rc != BS_OK) return rc;
  uint8_t* wsb = (uint8_t*)ws;
  rc = bs::launch_fill_rows((const int2*)(wsb + L.fill_off), (int)tb.fill.size(), tb.max_fill_rows,
                            dK, dV, nullptr, shape->n_kv_heads, shape->head_dim,
                            shape->kv_row_stride, 0, st);
  if (rc != BS_OK) return rc;
  if (tb.items.empty()) return BS_OK;

  BwdParams p;
  p.sv = bs::make_sched_view(wsb, L, tb, shape->n_kv_heads);
  p.n_kv_heads = shape->n_kv_heads;
  p.group = shape->n_q_heads / shape->n_kv_heads;
  p.q_rows = shape->q_rows;
  p.scale = shape->softmax_scale > 0.f ? shape->softmax_scale : 1.f / sqrtf((float)D);
  p.scale_log2 = p.scale * 1.4426950408889634f;
  p.LSE = LSE_final;
  p.delta = delta;
  p.lse_head_stride = shape->lse_head_stride;
  p.dK = (__nv_bfloat16*)dK;
  p.dV = (__nv_bfloat16*)dV;
  p.kv_row_stride = shape->kv_row_stride;
  p.dQ_acc = dQ_acc;
  p.n_q_heads = shape->n_q_heads;
  const int grid = tb.n_units < bs::sm_count() ? tb.n_units : bs::sm_count();
  if (D == 128) {
    rc = bs::set_max_smem_once((const void*)attn_bwd_kernel<128>, BwdSmem<128>::kBytes, 2);
    if (rc != BS_OK) return rc;
    attn_bwd_kernel<128><<<grid, kBwdThreads, BwdSmem<128>::kBytes, st>>>(tmQ, tmK, tmV, tmDO, tmDQ, tmDK, tmDV, p);
  } else {
    rc = bs::set_max_smem_once((const void*)attn_bwd_kernel<64>, BwdSmem<64>::kBytes, 3);
    if (rc != BS_OK) return rc;
    attn_bwd_kernel<64><<<grid, kBwdThreads, BwdSmem<64>::kBytes, st>>>(tmQ, tmK, tmV, tmDO, tmDQ, tmDK, tmDV, p);
  }
  BS_CUDA(cudaGetLastError());
  bs::count_launch();
  return BS_OK;
}
