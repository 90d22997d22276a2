// attn_fwd.cu — bs_attn_fwd: one Q-chunk x KV-chunk step of packed varlen / zigzag-CP causal
// attention on sm_100a (SURVEY.md 8(a) a2+a3; flash attention = exact attention).
//
// Kernel shape (one persistent CTA per SM, 384 threads, registers re-split by setmaxnreg):
//   warps 0-3  softmax warpgroup of Q tile 0   (thread r <-> row r of the 128-row tile)
//   warps 4-7  softmax warpgroup of Q tile 1
//   warp  8    MMA issuer (one elected lane): tcgen05.mma, accumulators in TMEM
//   warp  9    TMA producer: Q per item and tile, K/V blocks through a 4-stage smem ring
// A work item is (up to 256 query rows = two 128-row tiles of one query range, one query head).
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,256+D) O1 [384,384+D); P (bf16) overwrites
// the first 64 columns of its S.  Per KV block the tensor pipe runs, in issue order,
//   PV0(b) S0(b+1) PV1(b) S1(b+1)
// so that the softmax of one tile overlaps the MMAs of the other.  Softmax is fp32 with exp2,
// a lazily updated running max (rescale of O only when the max grew by more than 2^8) and the
// row sum kept in fp32; O is normalised and written as bf16 with LSE = m ln2 + ln l at the end.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include "common.h"
#include "launch_utils.h"
#include "ptx.cuh"
#include "sched.cuh"
#include "worklist.h"

namespace {

using namespace bs;
using namespace bs::ptx;

constexpr int kFwdThreads = 384;      // 2 softmax warpgroups + 1 auxiliary warpgroup (MMA, TMA)
constexpr int kRegsSoftmax = 208;     // setmaxnreg budgets: 256 * 208 + 128 * 88 = 384 * 168
constexpr int kRegsAux = 88;
constexpr int kStages = 4;              // K/V ring depth (K and V blocks alternate in the ring)
constexpr float kRescaleThreshold = 8.f;  // log2 units

struct FwdParams {
  SchedView sv;     // units = query items x n_q_heads
  int32_t n_q_heads, group;  // group = Hq / Hkv
  int32_t q_rows;
  float scale_log2;  // softmax_scale * log2(e)
  __nv_bfloat16* O;
  float* LSE;
  int64_t o_row_stride, lse_head_stride;
};

template <int D>
struct FwdSmem {
  static constexpr int kTileBytes = kTile * D * 2;  // one 128-row tile of Q, K or V
  static constexpr int kQOff = 0;                   // 2 Q tiles
  static constexpr int kKVOff = 2 * kTileBytes;     // kStages K/V tiles
  static constexpr int kBarOff = kKVOff + kStages * kTileBytes;
  // barriers: q_full[2], q_empty[2], kv_full[S], kv_empty[S], s_full[2], p_full[2], o_full[2]
  static constexpr int kNumBars = 4 + 2 * kStages + 6;
  static constexpr int kTmemSlotOff = kBarOff + kNumBars * 8;
  static constexpr int kSchedOff = kTmemSlotOff + 8;  // SchedRing of the dynamic scheduler
  static constexpr int kBytes = kSchedOff + 64;
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
// tile has a visible pair in it; tile t takes part in the block iff active(t).
struct Walker {
  const Span* spans;
  int n_spans, s, j, nb[2], at0[2], rows[2];
  Span sp;
  __device__ __forceinline__ void load_span() {
    while (s < n_spans) {
      sp = spans[s];
      nb[0] = span_blocks(at0[0], rows[0], sp);
      nb[1] = span_blocks(at0[1], rows[1], sp);
      if (max(nb[0], nb[1]) > 0) break;
      ++s;
    }
    j = 0;
  }
  __device__ __forceinline__ void init(const Span* sp_table, const Item& it) {
    spans = sp_table + it.span_begin;
    n_spans = it.n_spans;
    for (int t = 0; t < 2; ++t) {
      at0[t] = it.local0 + t * kTile;
      rows[t] = max(0, min(kTile, it.range_len - at0[t]));
    }
    s = 0;
    load_span();
  }
  __device__ __forceinline__ bool done() const { return s >= n_spans; }
  __device__ __forceinline__ bool active(int t) const { return j < nb[t]; }
  __device__ __forceinline__ void next() {
    if (++j >= max(nb[0], nb[1])) {
      ++s;
      load_span();
    }
  }
  // total blocks tile t takes part in over the whole item
  __device__ __forceinline__ int total(int t) const {
    int n = 0;
    for (int q = 0; q < n_spans; ++q) n += span_blocks(at0[t], rows[t], spans[q]);
    return n;
  }
};

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
template <int D>
__device__ __forceinline__ void issue_pv(uint32_t tmem_o, uint32_t tmem_p, uint32_t v_addr,
                                         bool accumulate) {
  constexpr uint32_t idesc = umma_idesc_bf16(kTile, D, 0, 1);  // B = V is MN-major (d contiguous)
#pragma unroll
  for (int kk = 0; kk < kTile / 16; ++kk) {
    // 16 keys = 16 rows of 128 B; the second 64-wide d half (D = 128) is one box (16 KB) further
    umma_ts(tmem_o, tmem_p + kk * 8, umma_desc_sw128(v_addr + kk * 2048, kTile * 128, 1024), idesc,
            accumulate || kk > 0);
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
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ FwdParams p) {
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
  uint64_t* p_full = s_full + 2;
  uint64_t* o_full = p_full + 2;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kTmemSlotOff);
  SchedRing* sched = reinterpret_cast<SchedRing*>(smem + L::kSchedOff);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 9 && lane == 0) {
    sched_ring_init(sched, 2 * kTile + 1);  // consumers: 256 softmax threads + the MMA lane
    for (int t = 0; t < 2; ++t) {
      mbar_init(&q_full[t], 1);
      mbar_init(&q_empty[t], 1);
      mbar_init(&s_full[t], 1);
      mbar_init(&p_full[t], kTile);
      mbar_init(&o_full[t], 1);
    }
    for (int i = 0; i < kStages; ++i) {
      mbar_init(&kv_full[i], 1);
      mbar_init(&kv_empty[i], 1);
    }
    fence_barrier_init();
    prefetch_tensormap(&tmQ);
    prefetch_tensormap(&tmK);
    prefetch_tensormap(&tmV);
  }
  if (warp == 8) tmem_alloc<512>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t smem_q = smem_u32(smem + L::kQOff), smem_kv = smem_u32(smem + L::kKVOff);

  if (warp >= 8) {
    setmaxnreg_dec<kRegsAux>();
    if (warp == 9 && lane == 0) {
      // ===================================== TMA producer =====================================
      uint32_t q_ph[2] = {0, 0};
      Ring ring;
      UnitProducer prod{sched};
      int32_t w;
      while ((w = prod.next(p.sv)) >= 0) {
        const Unit u = decode_unit(p.sv, w);
        const Item& it = u.item;
        const int h = u.head, g = h / p.group;
        Walker wk;
        wk.init(p.sv.spans, it);
        if (wk.done()) continue;
        // the first K/V block goes out before the Q tiles: the ring usually has room while the
        // Q buffers are still held by the previous unit's last S MMAs
        for (bool first = true; !wk.done(); wk.next(), first = false) {
          const int krow = wk.sp.begin + wk.j * kTile;
          for (int kv = 0; kv < 2; ++kv) {
            mbar_wait(&kv_empty[ring.stage], ring.phase ^ 1);
            mbar_arrive_expect_tx(&kv_full[ring.stage], L::kTileBytes);
            for (int half = 0; half < D / 64; ++half)
              tma_load_3d(smem + L::kKVOff + ring.stage * L::kTileBytes + half * (kTile * 128),
                          kv == 0 ? &tmK : &tmV, &kv_full[ring.stage], half * 64, g, krow);
            ring.advance();
          }
          if (first) {
            for (int t = 0; t < 2; ++t) {
              if (wk.total(t) == 0) continue;
              mbar_wait(&q_empty[t], q_ph[t] ^ 1);
              q_ph[t] ^= 1;
              mbar_arrive_expect_tx(&q_full[t], L::kTileBytes);
              for (int half = 0; half < D / 64; ++half)
                tma_load_3d(smem + L::kQOff + t * L::kTileBytes + half * (kTile * 128), &tmQ,
                            &q_full[t], half * 64, h, it.row0 + t * kTile);
            }
          }
        }
      }
    } else if (warp == 8 && lane == 0) {
      // ====================================== MMA issuer ======================================
      uint32_t q_ph[2] = {0, 0}, p_ph[2] = {0, 0};
      Ring ring;
      UnitConsumer cons{sched};
      int32_t w;
      while ((w = cons.next()) >= 0) {
        const Unit u = decode_unit(p.sv, w);
        const Item& it = u.item;
        Walker cur;
        cur.init(p.sv.spans, it);
        if (cur.done()) continue;
        const int tot[2] = {cur.total(0), cur.total(1)};
        int n_s[2] = {0, 0}, n_pv[2] = {0, 0};
        // S_t = Q_t K^T of one block; the first one of an item waits for the tile's Q, the last
        // one releases the tile's Q buffer to the producer (next item's Q streams in early)
        auto issue_s = [&](int t, uint32_t k_stage) {
          if (n_s[t] == 0) {
            mbar_wait(&q_full[t], q_ph[t]);
            q_ph[t] ^= 1;
            tc_fence_after();
          }
          issue_qk<D>(tmem + t * kTile, smem_q + t * L::kTileBytes,
                      smem_kv + k_stage * L::kTileBytes);
          tc_commit(&s_full[t]);
          if (++n_s[t] == tot[t]) tc_commit(&q_empty[t]);
        };
        // prologue: S_t(0)
        mbar_wait(&kv_full[ring.stage], ring.phase);
        tc_fence_after();
        for (int t = 0; t < 2; ++t)
          if (cur.active(t)) issue_s(t, ring.stage);
        tc_commit(&kv_empty[ring.stage]);
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
          for (int t = 0; t < 2; ++t) {
            if (cur.active(t)) {
              mbar_wait(&p_full[t], p_ph[t]);
              p_ph[t] ^= 1;
              tc_fence_after();
              issue_pv<D>(tmem + 256 + t * kTile, tmem + t * kTile,
                          smem_kv + v_stage * L::kTileBytes, n_pv[t] > 0);
              if (++n_pv[t] == tot[t]) tc_commit(&o_full[t]);
            }
            if (has_next && nxt.active(t)) issue_s(t, k_stage);
          }
          tc_commit(&kv_empty[v_stage]);
          if (!has_next) break;
          tc_commit(&kv_empty[k_stage]);
          cur = nxt;
        }
      }
    }
  } else {
    // ================================== softmax warpgroups ==================================
    setmaxnreg_inc<kRegsSoftmax>();
    const int t = warp >> 2;            // Q tile of this warpgroup
    const int r = threadIdx.x & 127;    // row of the tile owned by this thread
    const uint32_t lane_addr = uint32_t((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + lane_addr + t * kTile;        // S_t, and P_t over its first 64 cols
    const uint32_t tO = tmem + lane_addr + 256 + t * kTile;  // O_t
    const float2 sc2 = make_float2(p.scale_log2, p.scale_log2);
    uint32_t s_ph = 0, o_ph = 0;
    UnitConsumer cons{sched};
    int32_t w;
    while ((w = cons.next()) >= 0) {
      const Unit u = decode_unit(p.sv, w);
      const Item& it = u.item;
      const int h = u.head;
      Walker wk;
      wk.init(p.sv.spans, it);
      const int at0 = wk.at0[t];
      const bool valid = r < wk.rows[t];
      const int64_t grow = (int64_t)it.row0 + t * kTile + r;
      __nv_bfloat16* o_ptr = p.O + grow * p.o_row_stride + (int64_t)h * D;
      const int tot = wk.total(t);
      if (tot == 0) {  // no key of this call is visible to any row of the tile
        if (valid) {
          for (int c = 0; c < D / 8; ++c) reinterpret_cast<uint4*>(o_ptr)[c] = make_uint4(0, 0, 0, 0);
          p.LSE[(int64_t)h * p.lse_head_stride + grow] = -CUDART_INF_F;
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
        tc_fence_after();
        float s[kTile];
        tmem_ld32(tS, reinterpret_cast<uint32_t*>(s));
        tmem_ld32(tS + 32, reinterpret_cast<uint32_t*>(s) + 32);
        tmem_ld32(tS + 64, reinterpret_cast<uint32_t*>(s) + 64);
        tmem_ld32(tS + 96, reinterpret_cast<uint32_t*>(s) + 96);
        tmem_wait_ld();
        const int b0 = wk.j * kTile;
        if (b0 + kTile - 1 > at0 + wk.sp.off || b0 + kTile > wk.sp.len) {
          const int lim = min(at0 + r + wk.sp.off, wk.sp.len - 1) - b0;  // last visible column
#pragma unroll
          for (int c = 0; c < kTile; ++c)
            if (c > lim) s[c] = -CUDART_INF_F;
        }
        float mx0 = fmax3(s[0], s[1], s[2]), mx1 = fmax3(s[3], s[4], s[5]);
        float mx2 = fmax3(s[6], s[7], s[8]), mx3 = fmax3(s[9], s[10], s[11]);
#pragma unroll
        for (int c = 12; c < 124; c += 8) {
          mx0 = fmax3(mx0, s[c], s[c + 1]);
          mx1 = fmax3(mx1, s[c + 2], s[c + 3]);
          mx2 = fmax3(mx2, s[c + 4], s[c + 5]);
          mx3 = fmax3(mx3, s[c + 6], s[c + 7]);
        }
        mx0 = fmax3(mx0, s[124], s[125]);
        mx1 = fmax3(mx1, s[126], s[127]);
        const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * p.scale_log2;
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
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld32(tO + c * 32, o);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st32(tO + c * 32, o);
          }
        }
        const float neg_m = (m_used == -CUDART_INF_F) ? 0.f : -m_used;
        const float2 nm2 = make_float2(neg_m, neg_m);
#pragma unroll
        for (int c = 0; c < kTile / 32; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const float2 x = fma2(make_float2(s[c * 32 + 2 * i], s[c * 32 + 2 * i + 1]), sc2, nm2);
            const float2 e = make_float2(ex2(x.x), ex2(x.y));
            l2 = add2(l2, e);
            pk[i] = pack_bf16(e.x, e.y);
          }
          tmem_st16(tS + c * 16, pk);
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(&p_full[t]);
        ++cnt;
      }
      // ------------------------------------ epilogue ------------------------------------
      const float l = l2.x + l2.y;
      mbar_wait(&o_full[t], o_ph);
      o_ph ^= 1;
      tc_fence_after();
      const float inv_l = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(tO + c * 32, o);
        tmem_wait_ld();
        if (valid) {
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            uint4 pk;
            pk.x = pack_bf16(__uint_as_float(o[8 * v + 0]) * inv_l, __uint_as_float(o[8 * v + 1]) * inv_l);
            pk.y = pack_bf16(__uint_as_float(o[8 * v + 2]) * inv_l, __uint_as_float(o[8 * v + 3]) * inv_l);
            pk.z = pack_bf16(__uint_as_float(o[8 * v + 4]) * inv_l, __uint_as_float(o[8 * v + 5]) * inv_l);
            pk.w = pack_bf16(__uint_as_float(o[8 * v + 6]) * inv_l, __uint_as_float(o[8 * v + 7]) * inv_l);
            reinterpret_cast<uint4*>(o_ptr)[c * 4 + v] = pk;
          }
        }
      }
      if (valid)
        p.LSE[(int64_t)h * p.lse_head_stride + grow] =
            l > 0.f ? m_used * 0.69314718055994531f + __logf(l) : -CUDART_INF_F;
      tc_fence_before();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc<512>(tmem);
}

}  // namespace

namespace bs {

// Upload [header | items | spans | fill] into the workspace with one pageable-memory copy.
bs_status_t upload_tables(const SchedTables& tb, void* ws, size_t ws_bytes, cudaStream_t st,
                          WsLayout* layout) {
  const WsLayout L = ws_layout(tb.items.size(), tb.spans.size(), tb.groups.size(), tb.fill.size());
  BS_REQUIRE(ws != nullptr && ((uintptr_t)ws & 255) == 0, BS_ERR_WORKSPACE,
             "workspace is null or not 256-byte aligned");
  BS_REQUIRE(ws_bytes >= L.total, BS_ERR_WORKSPACE, "workspace too small: %zu < %zu bytes",
             ws_bytes, L.total);
  std::vector<uint8_t> blob;
  try {
    blob.assign(L.total, 0);
  } catch (const std::bad_alloc&) {
    return fail(BS_ERR_HOST_OOM, "out of host memory staging the work list");
  }
  SchedHeader* hd = reinterpret_cast<SchedHeader*>(blob.data());
  hd->counter = 0;
  hd->n_items = (int32_t)tb.items.size();
  hd->n_spans = (int32_t)tb.spans.size();
  hd->n_fill = (int32_t)tb.fill.size();
  hd->n_groups = (int32_t)tb.groups.size();
  hd->n_units = tb.n_units;
  if (!tb.groups.empty())
    memcpy(blob.data() + L.groups_off, tb.groups.data(), tb.groups.size() * sizeof(Group));
  if (!tb.items.empty())
    memcpy(blob.data() + L.items_off, tb.items.data(), tb.items.size() * sizeof(Item));
  if (!tb.spans.empty())
    memcpy(blob.data() + L.spans_off, tb.spans.data(), tb.spans.size() * sizeof(Span));
  if (!tb.fill.empty())
    memcpy(blob.data() + L.fill_off, tb.fill.data(), tb.fill.size() * sizeof(RowRange));
  BS_CUDA(cudaMemcpyAsync(ws, blob.data(), L.total, cudaMemcpyHostToDevice, st));
  *layout = L;
  return BS_OK;
}

int sm_count() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
      n = 148;
  }
  return n;
}

}  // namespace bs

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
                        void* stream) {
  bs_status_t rc = bs::validate_shape(shape, "bs_attn_fwd");
  if (rc != BS_OK) return rc;
  BS_REQUIRE(Q && K && V && O && LSE, BS_ERR_INVALID_ARG, "bs_attn_fwd: null tensor pointer");
  BS_REQUIRE(n_segs >= 0 && (segs || n_segs == 0), BS_ERR_INVALID_ARG, "bs_attn_fwd: bad segs");
  BS_REQUIRE(0 <= out_row_begin && out_row_begin <= out_row_end && out_row_end <= shape->q_rows,
             BS_ERR_INVALID_ARG, "bs_attn_fwd: output rows [%d,%d) outside [0,%d)", out_row_begin,
             out_row_end, shape->q_rows);
  BS_REQUIRE(((uintptr_t)O & 15) == 0, BS_ERR_INVALID_ARG, "bs_attn_fwd: O not 16-byte aligned");
  if (out_row_end == out_row_begin) return BS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  bs::SchedTables tb;
  rc = bs::build_fwd_tables(segs, n_segs, shape->q_rows, shape->kv_rows, out_row_begin, out_row_end,
                            shape->n_q_heads, &tb);
  if (rc != BS_OK) return rc;
  bs::WsLayout L;
  rc = bs::upload_tables(tb, ws, ws_bytes, st, &L);
  if (rc != BS_OK) return rc;
  uint8_t* wsb = (uint8_t*)ws;
  rc = bs::launch_fill_rows((const int2*)(wsb + L.fill_off), (int)tb.fill.size(), tb.max_fill_rows,
                            O, nullptr, LSE, shape->n_q_heads, shape->head_dim, shape->q_row_stride,
                            shape->lse_head_stride, st);
  if (rc != BS_OK) return rc;
  if (tb.items.empty()) return BS_OK;

  const int D = shape->head_dim;
  CUtensorMap tmQ, tmK, tmV;
  rc = bs::make_tensor_map_3d(&tmQ, Q, 2, D, shape->n_q_heads, shape->q_rows, shape->q_row_stride,
                              64, bs::kTile, true);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmK, K, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, true);
  if (rc != BS_OK) return rc;
  rc = bs::make_tensor_map_3d(&tmV, V, 2, D, shape->n_kv_heads, shape->kv_rows,
                              shape->kv_row_stride, 64, bs::kTile, true);
  if (rc != BS_OK) return rc;

  FwdParams p;
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
    BS_CUDA(cudaFuncSetAttribute(attn_fwd_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 FwdSmem<128>::kAlloc));
    attn_fwd_kernel<128><<<grid, kFwdThreads, FwdSmem<128>::kAlloc, st>>>(tmQ, tmK, tmV, p);
  } else {
    BS_CUDA(cudaFuncSetAttribute(attn_fwd_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 FwdSmem<64>::kAlloc));
    attn_fwd_kernel<64><<<grid, kFwdThreads, FwdSmem<64>::kAlloc, st>>>(tmQ, tmK, tmV, p);
  }
  BS_CUDA(cudaGetLastError());
  bs::count_launch();
  return BS_OK;
}

}  // extern "C"
