// sched.cuh — device side of the persistent tile scheduler: one warp of the CTA
// pulls unit indices from the global atomic cursor and hands them to the other warps through a
// two-slot shared-memory ring, so every role of a warp-specialised kernel walks the same units.
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
  int32_t n_groups, n_units, n_heads;
};

struct Unit {
  Item item;
  int32_t head;
};

// unit index -> (item, head): binary search of the group, then head-major inside the group.
__device__ __forceinline__ Unit decode_unit(const SchedView& sv, int32_t w) {
  int lo = 0, hi = sv.n_groups - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (sv.groups[mid].unit_begin <= w) lo = mid; else hi = mid - 1;
  }
  const Group g = sv.groups[lo];
  const int local = w - g.unit_begin;
  Unit u;
  u.head = local / g.n_items;
  u.item = sv.items[g.item_begin + local % g.n_items];
  return u;
}

constexpr int kSchedSlots = 2;

struct SchedRing {  // lives in shared memory
  uint64_t full[kSchedSlots], empty[kSchedSlots];
  int32_t unit[kSchedSlots];
};

// n_consumers = threads that call UnitConsumer::next()
__device__ __forceinline__ void sched_ring_init(SchedRing* r, uint32_t n_consumers) {
  for (int i = 0; i < kSchedSlots; ++i) {
    ptx::mbar_init(&r->full[i], 1);
    ptx::mbar_init(&r->empty[i], n_consumers);
  }
}

struct UnitProducer {  // one thread
  SchedRing* r;
  uint32_t n = 0;
  // Returns the next unit index of this CTA, or -1 when the cursor ran out (also published).
  __device__ __forceinline__ int32_t next(const SchedView& sv) {
    int32_t w = atomicAdd(sv.counter, 1);
    if (w >= sv.n_units) w = -1;
    const uint32_t slot = n % kSchedSlots, ph = (n / kSchedSlots) & 1;
    ptx::mbar_wait(&r->empty[slot], ph ^ 1);
    r->unit[slot] = w;
    ptx::mbar_arrive(&r->full[slot]);
    ++n;
    return w;
  }
};

// Tell the compiler that a value is the same in every lane of a converged warp (it then keeps
// it, and what is computed from it, in uniform registers - e.g. the tcgen05.mma descriptors).
template <class T>
__device__ __forceinline__ T warp_uniform(T v) {
  return __shfl_sync(0xffffffffu, v, 0);
}

struct UnitConsumer {  // every consuming thread
  SchedRing* r;
  uint32_t n = 0;
  __device__ __forceinline__ int32_t next() {
    const uint32_t slot = n % kSchedSlots, ph = (n / kSchedSlots) & 1;
    ptx::mbar_wait(&r->full[slot], ph);
    const int32_t w = r->unit[slot];
    ptx::mbar_arrive(&r->empty[slot]);
    ++n;
    return w;
  }
  // Whole converged warp consumes as ONE consumer (one arrival on the empty barrier).
  __device__ __forceinline__ int32_t next_warp() {
    const uint32_t slot = n % kSchedSlots, ph = (n / kSchedSlots) & 1;
    ptx::mbar_wait_warp(&r->full[slot], ph);
    const int32_t w = warp_uniform(r->unit[slot]);
    __syncwarp();
    if (ptx::elect_one()) ptx::mbar_arrive(&r->empty[slot]);
    ++n;
    return w;
  }
};

// decode_unit for a converged warp: every lane loads the same words; the fields come back uniform.
__device__ __forceinline__ Unit decode_unit_warp(const SchedView& sv, int32_t w) {
  Unit u = decode_unit(sv, w);
  u.head = warp_uniform(u.head);
  u.item.row0 = warp_uniform(u.item.row0);
  u.item.local0 = warp_uniform(u.item.local0);
  u.item.range_len = warp_uniform(u.item.range_len);
  u.item.span_begin = warp_uniform(u.item.span_begin);
  u.item.n_spans = warp_uniform(u.item.n_spans);
  return u;
}

}  // namespace bs
