// sched.cuh — device side of the persistent tile scheduler: a scheduler warp of
// the CTA pulls unit indices from the global atomic cursor, decodes them and hands them to the
// other warps through a small shared-memory ring, so that every role of a warp-specialised
// kernel walks the same units and the cursor / table latency (several microseconds of dependent
// L2 round trips) stays off the critical path of short units.
// The cursor order is the host's longest-first / locality order (worklist.h).
#pragma once
#include "ptx.cuh"
#include "worklist.h"

namespace bs {

struct SchedView {  // device pointers into the uploaded workspace
  int32_t* counter;
  const Item* items;
  const Span* spans;
  const Group* groups;
  const CUtensorMap* tmaps;  // clipped tensor maps of ragged range ends (worklist.h), 128-byte aligned
  int32_t n_groups, n_units, n_heads;
  int32_t n_span_clips;      // bwd: the K / V maps of the item clips follow 2 * n_span_clips Q / dO maps
  int32_t n_item_clips;
};

struct Unit {
  Item item;
  int32_t head;
  Span sp[2];  // the item's first two spans (most items have one or two): the consumers' walkers
               // start from registers instead of a dependent global load at every unit start
};
// span s of a unit: cached copy or the global table
__device__ __forceinline__ Span unit_span(const Unit& u, const Span* table, int s) {
  if (s == 0) return u.sp[0];
  if (s == 1) return u.sp[1];
  return table[u.item.span_begin + s];
}

// unit index -> (item, head): find the group (a CTA's unit indices only grow, so the search
// walks forward from the group of its previous unit: *hint), then head-major inside the group.
__device__ __forceinline__ Unit decode_unit(const SchedView& sv, int32_t w, int32_t* hint) {
  int lo = *hint;
  while (lo + 1 < sv.n_groups && sv.groups[lo + 1].unit_begin <= w) ++lo;
  *hint = lo;
  const Group g = sv.groups[lo];
  const int local = w - g.unit_begin;
  Unit u;
  u.head = local / g.n_items;
  u.item = sv.items[g.item_begin + local % g.n_items];
  u.sp[0] = sv.spans[u.item.span_begin];
  u.sp[1] = u.item.n_spans > 1 ? sv.spans[u.item.span_begin + 1] : u.sp[0];
  return u;
}

// kSlots = depth of the ring = how far the scheduler warp may run ahead of the slowest role.  A
// claimed unit cannot move to another CTA any more, so less look-ahead means later binding and a
// better balance; measured on cfg2 (3 -> 2 -> 1 slots): forward 0.695 -> 0.688 -> 0.692 ms,
// backward 1.569 -> 1.549 -> 1.517 ms; 4 slots are slower than 3 in both.  The kernels choose.
template <int kSlots>
struct SchedRingT {  // lives in shared memory (16-byte aligned)
  Item item[kSlots];  // decoded by the producer: consumers never touch the global tables
  Span sp[kSlots][2];
  int32_t head[kSlots];
  int32_t unit[kSlots];
  uint64_t full[kSlots], empty[kSlots];
  static constexpr int kBytes = 128 * kSlots;
};

// n_consumers = arrivals per slot on the empty barrier (threads calling next(), warps calling
// next_warp())
template <int kSlots>
__device__ __forceinline__ void sched_ring_init(SchedRingT<kSlots>* r, uint32_t n_consumers) {
  static_assert(sizeof(SchedRingT<kSlots>) <= SchedRingT<kSlots>::kBytes, "SchedRing size");
  for (int i = 0; i < kSlots; ++i) {
    ptx::mbar_init(&r->full[i], 1);
    ptx::mbar_init(&r->empty[i], n_consumers);
  }
}

template <int kSlots>
struct UnitProducerT {  // one thread (the scheduler warp's lane 0)
  SchedRingT<kSlots>* r;
  uint32_t n = 0;
  int32_t hint = 0, last = 0;
  // Pulls the next unit of this CTA from the global cursor, decodes it and publishes it.
  // Returns false when the cursor ran out (also published, as unit -1).
  // Look-ahead: up to kSlots - 1 units beyond the one the slowest consumer works on while
  // plenty of units are left; once the cursor is within 4 rounds of the end a unit is only
  // claimed when every consumer has taken the previous one, so that the short tail units go to
  // whichever CTA is free first (greedy longest-first).
  __device__ __forceinline__ bool next(const SchedView& sv, Unit* u) {
    if (n > 0 && last >= sv.n_units - 4 * (int32_t)gridDim.x) {
      const uint32_t pslot = (n - 1) % kSlots, pph = ((n - 1) / kSlots) & 1;
      ptx::mbar_wait(&r->empty[pslot], pph);
    }
    int32_t w = atomicAdd(sv.counter, 1);
    last = w;
    if (w >= sv.n_units) w = -1;
    if (w >= 0) *u = decode_unit(sv, w, &hint);
    const uint32_t slot = n % kSlots, ph = (n / kSlots) & 1;
    ptx::mbar_wait(&r->empty[slot], ph ^ 1);
    if (w >= 0) {
      r->item[slot] = u->item;
      r->head[slot] = u->head;
      r->sp[slot][0] = u->sp[0];
      r->sp[slot][1] = u->sp[1];
    }
    r->unit[slot] = w;
    ptx::mbar_arrive(&r->full[slot]);
    ++n;
    return w >= 0;
  }
};

// Tell the compiler that a value is the same in every lane of a converged warp (it then keeps
// it, and what is computed from it, in uniform registers - e.g. the tcgen05.mma descriptors).
template <class T>
__device__ __forceinline__ T warp_uniform(T v) {
  return __shfl_sync(0xffffffffu, v, 0);
}

template <int kSlots>
struct UnitConsumerT {  // every consuming thread
  SchedRingT<kSlots>* r;
  uint32_t n = 0;
  __device__ __forceinline__ bool next(Unit* u) {
    const uint32_t slot = n % kSlots, ph = (n / kSlots) & 1;
    ptx::mbar_wait(&r->full[slot], ph);
    const int32_t w = r->unit[slot];
    if (w >= 0) {
      u->item = r->item[slot];
      u->head = r->head[slot];
      u->sp[0] = r->sp[slot][0];
      u->sp[1] = r->sp[slot][1];
    }
    ptx::mbar_arrive(&r->empty[slot]);
    ++n;
    return w >= 0;
  }
  // Warp-collective form for the lanes in `mask` (all of them call it, converged): lane `leader`
  // alone polls the slot's barrier and releases the slot; the others park at the warp barrier.
  // For roles that run far ahead of the pipeline and would otherwise have 32 lanes polling a
  // barrier for the length of a unit - shared-memory polls that the tensor core's operand reads
  // and the other warps of the scheduler partition pay for (measured: 5-9 % of either kernel).
  __device__ __forceinline__ bool next_warp(Unit* u, uint32_t mask, int leader) {
    const uint32_t slot = n % kSlots, ph = (n / kSlots) & 1;
    const bool lead = (threadIdx.x & 31) == leader;
    if (lead) ptx::mbar_wait(&r->full[slot], ph);
    __syncwarp(mask);
    const int32_t w = r->unit[slot];
    if (w >= 0) {
      u->item = r->item[slot];
      u->head = r->head[slot];
      u->sp[0] = r->sp[slot][0];
      u->sp[1] = r->sp[slot][1];
    }
    __syncwarp(mask);
    if (lead) ptx::mbar_arrive(&r->empty[slot]);
    ++n;
    return w >= 0;
  }
  // Converged warp, every lane waits for the slot itself (no extra hop on the way in), one
  // arrival per warp on the way out.
  __device__ __forceinline__ bool next_arrive_once(Unit* u) {
    const uint32_t slot = n % kSlots, ph = (n / kSlots) & 1;
    ptx::mbar_wait(&r->full[slot], ph);
    const int32_t w = r->unit[slot];
    if (w >= 0) {
      u->item = r->item[slot];
      u->head = r->head[slot];
      u->sp[0] = r->sp[slot][0];
      u->sp[1] = r->sp[slot][1];
    }
    __syncwarp();
    if ((threadIdx.x & 31) == 0) ptx::mbar_arrive(&r->empty[slot]);
    ++n;
    return w >= 0;
  }
  // Wait for slot n and read it without consuming it (lanes 1-31 of a warp whose lane 0
  // consumes for the warp afterwards).
  __device__ __forceinline__ void wait_peek(Unit* u) const {
    const uint32_t slot = n % kSlots, ph = (n / kSlots) & 1;
    ptx::mbar_wait(&r->full[slot], ph);
    u->item = r->item[slot];
    u->head = r->head[slot];
    u->sp[0] = r->sp[slot][0];
    u->sp[1] = r->sp[slot][1];
  }
};

}  // namespace bs
