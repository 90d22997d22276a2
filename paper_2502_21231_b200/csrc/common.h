// common.h — error reporting and launch accounting shared by the library's translation units.
#pragma once
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "bytescale_attn.h"

namespace bs {

// Thread-local detail text returned by bs_last_error().
bs_status_t fail(bs_status_t code, const char* fmt, ...);
void count_launch(int n = 1);

}  // namespace bs

#define BS_REQUIRE(cond, code, ...)                      \
  do {                                                   \
    if (!(cond)) return ::bs::fail((code), __VA_ARGS__); \
  } while (0)

#define BS_CUDA(expr)                                                                         \
  do {                                                                                        \
    cudaError_t e__ = (expr);                                                                 \
    if (e__ != cudaSuccess)                                                                   \
      return ::bs::fail(BS_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e__));        \
  } while (0)
