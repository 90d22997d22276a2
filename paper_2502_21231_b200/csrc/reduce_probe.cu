// reduce_probe.cu — bs_reduce_probe: measurement aid for the backward's roofline.
//
// bs_attn_bwd adds every 128 x 128 tile-block's partial dQ (64 KB of fp32 at D = 128) into dQ_acc
// with TMA reduce-adds that execute in the L2 atomic units.  This kernel issues nothing but such
// reduce boxes - the same instruction, box shape (128 rows x 32 fp32, 128-byte swizzle) and
// tensor map the backward uses, two boxes in flight per CTA, one CTA per SM - so that bench.py
// can report the backward's reduction traffic against what the device sustains when nothing else
// runs (on a B200 that ceiling, ~12 B/clk per SM with all SMs active,
// is what bounds the backward's steady state, not the tensor pipe).
#include <cuda_runtime.h>

#include "common.h"
#include "launch_utils.h"
#include "ptx.cuh"

namespace {

using namespace bs;
using namespace bs::ptx;

constexpr int kBoxBytes = kTile * 32 * 4;  // 16 KB
constexpr int kProbeThreads = 128;

__global__ void __launch_bounds__(kProbeThreads)
reduce_probe_kernel(const __grid_constant__ CUtensorMap tm, int n_row_tiles, int n_heads, int n_chunks,
                    int boxes) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  for (int i = threadIdx.x; i < 2 * kBoxBytes / 4; i += blockDim.x) reinterpret_cast<float*>(smem)[i] = 0.f;
  fence_proxy_async_smem();
  __syncthreads();
  if (threadIdx.x != 0) return;
  // the backward's order: the chunks of one (query tile, head) back to back, then another tile
  for (int b = 0; b < boxes; ++b) {
    const int it = b / n_chunks, c = b % n_chunks;
    const int tile = (int)(((unsigned)blockIdx.x * 131u + (unsigned)it * 7u) % (unsigned)n_row_tiles);
    const int h = (int)(((unsigned)blockIdx.x + (unsigned)it) % (unsigned)n_heads);
    bulk_wait_group_read<1>();  // the box two back has been read
    tma_reduce_add_3d(&tm, smem + (b & 1) * kBoxBytes, c * 32, h, tile * kTile);
    bulk_commit_group();
  }
  bulk_wait_group<0>();
}

}  // namespace

extern "C" bs_status_t bs_reduce_probe(float* acc, int32_t rows, int32_t n_heads, int32_t head_dim,
                                       int32_t boxes_per_cta, void* stream) {
  BS_REQUIRE(acc != nullptr && ((uintptr_t)acc & 15) == 0, BS_ERR_INVALID_ARG,
             "bs_reduce_probe: acc null or not 16-byte aligned");
  BS_REQUIRE(rows >= kTile && rows % kTile == 0 && n_heads >= 1 && head_dim >= 32 && head_dim % 32 == 0 &&
                 head_dim <= 256 && boxes_per_cta >= 0,
             BS_ERR_INVALID_ARG, "bs_reduce_probe: rows %d (multiple of 128), heads %d, head_dim %d "
             "(multiple of 32, <= 256), boxes %d", rows, n_heads, head_dim, boxes_per_cta);
  if (boxes_per_cta == 0) return BS_OK;
  bs_status_t rc = bs::check_device();
  if (rc != BS_OK) return rc;
  CUtensorMap tm;
  rc = bs::make_tensor_map_3d(&tm, acc, 4, head_dim, n_heads, rows, (int64_t)n_heads * head_dim, 32,
                              kTile, 128);
  if (rc != BS_OK) return rc;
  const int smem_bytes = 2 * kBoxBytes + 1024;
  rc = bs::set_max_smem_once((const void*)reduce_probe_kernel, smem_bytes, 8);
  if (rc != BS_OK) return rc;
  reduce_probe_kernel<<<bs::sm_count(), kProbeThreads, smem_bytes, (cudaStream_t)stream>>>(
      tm, rows / kTile, n_heads, head_dim / 32, boxes_per_cta);
  BS_CUDA(cudaGetLastError());
  bs::count_launch();
  return BS_OK;
}
