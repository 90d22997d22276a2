// status.cpp — status strings, thread-local error text, launch counter.
#include <cstring>

#include "common.h"

namespace {
thread_local char g_err[512] = "";
thread_local int64_t g_launches = 0;
}  // namespace

namespace bs {
bs_status_t fail(bs_status_t code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
void count_launch(int n) { g_launches += n; }
}  // namespace bs

extern "C" {
const char* bs_status_string(bs_status_t s) {
  switch (s) {
    case BS_OK: return "BS_OK";
    case BS_ERR_INVALID_ARG: return "BS_ERR_INVALID_ARG";
    case BS_ERR_UNSUPPORTED: return "BS_ERR_UNSUPPORTED";
    case BS_ERR_WORKSPACE: return "BS_ERR_WORKSPACE";
    case BS_ERR_CUDA: return "BS_ERR_CUDA";
    case BS_ERR_HOST_OOM: return "BS_ERR_HOST_OOM";
  }
  return "BS_ERR_UNKNOWN";
}
const char* bs_last_error(void) { return g_err; }
int bs_version(void) { return BS_VERSION; }
int64_t bs_launch_count(void) { return g_launches; }
void bs_launch_count_reset(void) { g_launches = 0; }
}
