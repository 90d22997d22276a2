// trace.cuh — debug-only clock64() stamps of CTA 0 for the two attention kernels.
// Nothing of this exists in the product build: without -DBS_FWD_TRACE / -DBS_BWD_TRACE the macros
// expand to nothing and no symbol is exported.  A trace build (BS_NVCC_EXTRA=-DBS_BWD_TRACE
// python -m paper_2502_21231_b200.build --force) exports bs_debug_*_trace, which copy the
// stamps to the host; they are how the per-role timelines in DESIGN.md section 7 were measured.
// Include once per kernel translation unit, after defining BS_TRACE_KERNEL_FWD or _BWD.
#pragma once

#if defined(BS_TRACE_KERNEL_FWD) && defined(BS_FWD_TRACE)
__device__ long long g_fwd_trace[4][8][256];   // [role][event][block iteration]
__device__ long long g_fwd_utrace[5][8][64];   // [role][event][unit]
#define TRACE(role, ev, it)                                                    \
  do {                                                                         \
    if (blockIdx.x == 0 && (it) < 256) g_fwd_trace[role][ev][it] = clock64();  \
  } while (0)
#define UTRACE(t, ev, n)                                                       \
  do {                                                                         \
    if (blockIdx.x == 0 && (n) < 64) g_fwd_utrace[t][ev][n] = clock64();       \
  } while (0)
#define UTRACE_VALUE(t, ev, n, v)                                              \
  do {                                                                         \
    if (blockIdx.x == 0 && (n) < 64) g_fwd_utrace[t][ev][n] = (v);             \
  } while (0)
extern "C" int bs_debug_fwd_trace(long long* host_out) {
  return (int)cudaMemcpyFromSymbol(host_out, g_fwd_trace, sizeof(g_fwd_trace));
}
extern "C" int bs_debug_fwd_utrace(long long* host_out) {
  return (int)cudaMemcpyFromSymbol(host_out, g_fwd_utrace, sizeof(g_fwd_utrace));
}
#elif defined(BS_TRACE_KERNEL_BWD) && defined(BS_BWD_TRACE)
__device__ long long g_bwd_trace[3][10][512];  // [role][event][iteration]
#define TRACE(role, ev, it)                                                    \
  do {                                                                         \
    if (blockIdx.x == 0 && (it) < 512) g_bwd_trace[role][ev][it] = clock64();  \
  } while (0)
extern "C" int bs_debug_bwd_trace(long long* host_out) {
  return (int)cudaMemcpyFromSymbol(host_out, g_bwd_trace, sizeof(g_bwd_trace));
}
#endif

#ifndef TRACE
#define TRACE(role, ev, it) do {} while (0)
#endif
#ifndef UTRACE
#define UTRACE(t, ev, n) do {} while (0)
#define UTRACE_VALUE(t, ev, n, v) do {} while (0)
#endif
