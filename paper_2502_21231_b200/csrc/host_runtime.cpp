// host_runtime.cpp — host-side plumbing shared by the device entry points: the compute-capability
// check, the once-per-device kernel attribute, and the upload of the work-item tables through a
// library-owned ring of pinned staging buffers.
//
// Why a pinned ring: cudaMemcpyAsync from pageable memory is staged by the driver INSIDE the call
// and only after the stream's earlier work has drained far enough - the host would block behind
// the previous kernels on every bs_attn_fwd / bs_attn_bwd call, which the header rules out
// ("never synchronises the device").  From pinned memory the copy is a plain DMA enqueued on the
// caller's stream.  A slot is reused only after the copy that last read it has completed (one
// event per slot); with kSlots calls in flight the host waits for the oldest copy - bounded
// look-ahead, not a device synchronisation.
#include <cuda_runtime.h>

#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "launch_utils.h"

namespace bs {

namespace {
constexpr int kSlots = 64;
constexpr int kMaxDevices = 64;

struct Slot {
  uint8_t* host = nullptr;
  size_t cap = 0;
  cudaEvent_t done = nullptr;
  bool in_flight = false;
};
std::mutex g_mu;
Slot g_slots[kSlots];
size_t g_next = 0;

int g_cc[kMaxDevices];        // 0 = unknown, else major * 10 + minor
int g_sms[kMaxDevices];
uint32_t g_attr_done[kMaxDevices];  // bit k: kernel slot k has its shared-memory attribute
}  // namespace

bs_status_t check_device(int* device_out) {
  int dev = 0;
  BS_CUDA(cudaGetDevice(&dev));
  BS_REQUIRE(dev >= 0 && dev < kMaxDevices, BS_ERR_UNSUPPORTED, "device index %d", dev);
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_cc[dev] == 0) {
    int major = 0, minor = 0, sms = 0;
    BS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    BS_CUDA(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
    BS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    g_cc[dev] = major * 10 + minor;
    g_sms[dev] = sms > 0 ? sms : 148;
  }
  // the kernels are built for sm_100a only (tcgen05 / TMEM / TMA): architecture-specific code
  // runs on compute capability 10.0 and nothing else
  BS_REQUIRE(g_cc[dev] == 100, BS_ERR_UNSUPPORTED,
             "device %d has compute capability %d.%d; this library is built for sm_100a (B200)",
             dev, g_cc[dev] / 10, g_cc[dev] % 10);
  if (device_out) *device_out = dev;
  return BS_OK;
}

int sm_count() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return 148;
  std::lock_guard<std::mutex> lock(g_mu);
  return g_sms[dev] > 0 ? g_sms[dev] : 148;
}

bs_status_t set_max_smem_once(const void* func, int bytes, int kernel_slot) {
  int dev = 0;
  BS_CUDA(cudaGetDevice(&dev));
  BS_REQUIRE(dev >= 0 && dev < kMaxDevices && kernel_slot >= 0 && kernel_slot < 32,
             BS_ERR_UNSUPPORTED, "device index %d", dev);
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_attr_done[dev] & (1u << kernel_slot)) return BS_OK;
  BS_CUDA(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  g_attr_done[dev] |= 1u << kernel_slot;
  return BS_OK;
}

bs_status_t check_workspace(const SchedTables& tb, size_t tmap_bytes, const void* ws,
                            size_t ws_bytes, WsLayout* layout) {
  const WsLayout L = ws_layout(tb.items.size(), tb.spans.size(), tb.groups.size(), tb.fill.size(),
                               tmap_bytes);
  BS_REQUIRE(ws != nullptr && ((uintptr_t)ws & 255) == 0, BS_ERR_WORKSPACE,
             "workspace is null or not 256-byte aligned");
  BS_REQUIRE(ws_bytes >= L.total, BS_ERR_WORKSPACE, "workspace too small: %zu < %zu bytes",
             ws_bytes, L.total);
  *layout = L;
  return BS_OK;
}

bs_status_t append_clipped_maps(SchedTables* tb, size_t slot0, size_t slot_stride,
                                const std::vector<int32_t>& end_rows, const void* base,
                                int head_dim, int n_heads, int64_t row_stride_elems) {
  static_assert(sizeof(CUtensorMap) == kTensorMapBytes, "CUtensorMap size");
  try {
    const size_t need = (slot0 + (end_rows.empty() ? 0 : (end_rows.size() - 1) * slot_stride + 1)) *
                        kTensorMapBytes;
    if (tb->tmaps.size() < need) tb->tmaps.resize(need);
  } catch (const std::bad_alloc&) {
    return fail(BS_ERR_HOST_OOM, "out of host memory building the clipped tensor maps");
  }
  for (size_t i = 0; i < end_rows.size(); ++i) {
    CUtensorMap m;
    bs_status_t rc = make_tensor_map_3d(&m, base, 2, head_dim, n_heads, end_rows[i],
                                        row_stride_elems, 64, kTile, 128);
    if (rc != BS_OK) return rc;
    memcpy(tb->tmaps.data() + (slot0 + i * slot_stride) * kTensorMapBytes, &m, kTensorMapBytes);
  }
  return BS_OK;
}

// [header | items | spans | groups | fill | tensor maps] -> workspace, one DMA from a pinned slot.
bs_status_t upload_tables(const SchedTables& tb, const WsLayout& L, void* ws, cudaStream_t st) {
  std::lock_guard<std::mutex> lock(g_mu);
  Slot& s = g_slots[g_next];
  g_next = (g_next + 1) % kSlots;
  if (s.done == nullptr) BS_CUDA(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
  if (s.in_flight) {  // the copy that read this slot kSlots calls ago
    BS_CUDA(cudaEventSynchronize(s.done));
    s.in_flight = false;
  }
  if (s.cap < L.total) {
    if (s.host) BS_CUDA(cudaFreeHost(s.host));
    s.host = nullptr;
    s.cap = 0;
    size_t cap = 32 * 1024;
    while (cap < L.total) cap *= 2;
    void* p = nullptr;
    if (cudaHostAlloc(&p, cap, cudaHostAllocDefault) != cudaSuccess) {
      (void)cudaGetLastError();
      return fail(BS_ERR_HOST_OOM, "out of pinned host memory staging the work list (%zu bytes)", cap);
    }
    s.host = (uint8_t*)p;
    s.cap = cap;
  }
  memset(s.host, 0, L.total);
  SchedHeader* hd = reinterpret_cast<SchedHeader*>(s.host);
  hd->counter = 0;
  hd->n_items = (int32_t)tb.items.size();
  hd->n_spans = (int32_t)tb.spans.size();
  hd->n_fill = (int32_t)tb.fill.size();
  hd->n_groups = (int32_t)tb.groups.size();
  hd->n_units = tb.n_units;
  if (!tb.groups.empty())
    memcpy(s.host + L.groups_off, tb.groups.data(), tb.groups.size() * sizeof(Group));
  if (!tb.items.empty())
    memcpy(s.host + L.items_off, tb.items.data(), tb.items.size() * sizeof(Item));
  if (!tb.spans.empty())
    memcpy(s.host + L.spans_off, tb.spans.data(), tb.spans.size() * sizeof(Span));
  if (!tb.fill.empty())
    memcpy(s.host + L.fill_off, tb.fill.data(), tb.fill.size() * sizeof(RowRange));
  if (!tb.tmaps.empty()) memcpy(s.host + L.tmaps_off, tb.tmaps.data(), tb.tmaps.size());
  BS_CUDA(cudaMemcpyAsync(ws, s.host, L.total, cudaMemcpyHostToDevice, st));
  BS_CUDA(cudaEventRecord(s.done, st));
  s.in_flight = true;
  return BS_OK;
}

}  // namespace bs
