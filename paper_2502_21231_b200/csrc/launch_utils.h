// launch_utils.h — host-side helpers shared by the library's .cu files: shape validation,
// the uncovered-row fill launch, and TMA tensor-map creation through the driver entry point
// (so the library links against cudart only).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "common.h"

namespace bs {

bs_status_t validate_shape(const bs_attn_shape_t* s, const char* who);

// Zero rows [begin,end) of up to two [row][head][D] bf16 tensors and set lse[h][row] = -inf for
// each (begin,end) pair in the device array d_ranges.  max_rows = longest range (grid sizing).
bs_status_t launch_fill_rows(const int2* d_ranges, int n_ranges, int64_t max_rows, void* A, void* B,
                             float* lse, int n_heads, int head_dim, int64_t row_stride,
                             int64_t lse_head_stride, cudaStream_t st);

// 3-D tensor map over a [rows][heads][head_dim] tensor (innermost first: dim, head, row).
//   elem_bytes 2 (bf16) or 4 (fp32); box = (box_dim, 1, box_rows); swizzle: 0 (none), 64 or 128 bytes
//   (box_dim * elem_bytes must be 128) or none.
bs_status_t make_tensor_map_3d(CUtensorMap* map, const void* base, int elem_bytes, int head_dim,
                               int n_heads, int64_t rows, int64_t row_stride_elems, int box_dim,
                               int box_rows, int swizzle);

}  // namespace bs

#include "worklist.h"
namespace bs {
// host_runtime.cpp
// BS_ERR_UNSUPPORTED unless the current device is compute capability 10.0 (the kernels are sm_100a).
bs_status_t check_device(int* device_out = nullptr);
int sm_count();  // of the current device (after check_device)
// cudaFuncAttributeMaxDynamicSharedMemorySize, set once per device and kernel (kernel_slot < 32)
bs_status_t set_max_smem_once(const void* func, int bytes, int kernel_slot);
// Workspace checks (null / alignment / size) and layout; enqueues nothing.  tmap_bytes = size of
// the clipped tensor maps the entry point is going to put into tb.tmaps.
bs_status_t check_workspace(const SchedTables& tb, size_t tmap_bytes, const void* ws, size_t ws_bytes,
                            WsLayout* layout);
// Appends to tb->tmaps one tensor map per row in `end_rows`: the map of make_tensor_map_3d over
// the same tensor with its row extent cut at that row (TMA zero-fills the rows past it).
bs_status_t append_clipped_maps(SchedTables* tb, size_t slot0, size_t slot_stride,
                                const std::vector<int32_t>& end_rows, const void* base,
                                int head_dim, int n_heads, int64_t row_stride_elems);
// Tables -> workspace on `st` from a pinned staging slot (no stream synchronisation).
bs_status_t upload_tables(const SchedTables& tb, const WsLayout& layout, void* ws, cudaStream_t st);
}  // namespace bs

#include "sched.cuh"
namespace bs {
inline SchedView make_sched_view(uint8_t* ws, const WsLayout& L, const SchedTables& tb,
                                 int32_t n_heads) {
  SchedView sv;
  sv.counter = reinterpret_cast<int32_t*>(ws);
  sv.items = reinterpret_cast<const Item*>(ws + L.items_off);
  sv.spans = reinterpret_cast<const Span*>(ws + L.spans_off);
  sv.groups = reinterpret_cast<const Group*>(ws + L.groups_off);
  sv.tmaps = reinterpret_cast<const CUtensorMap*>(ws + L.tmaps_off);
  sv.n_span_clips = (int32_t)tb.clip_span_rows.size();
  sv.n_item_clips = (int32_t)tb.clip_item_rows.size();
  sv.n_groups = (int32_t)tb.groups.size();
  sv.n_units = tb.n_units;
  sv.n_heads = n_heads;
  return sv;
}
}  // namespace bs
