// attn_bwd.cu — bs_attn_bwd (placeholder while the tcgen05 backward kernel is brought up).
#include "common.h"
extern "C" bs_status_t bs_attn_bwd(const bs_attn_shape_t*, const void*, const void*, const void*,
                                   const void*, const float*, const float*, const bs_seg_t*,
                                   int32_t, float*, void*, void*, void*, size_t, void*) {
  return bs::fail(BS_ERR_UNSUPPORTED, "bs_attn_bwd: not built yet");
}
