// ws_util.cu -- status strings, version, error and launch bookkeeping of the C ABI (include/ws.h).
#include <atomic>

#include "ws_internal.h"

namespace {
thread_local int g_last_cuda_error = 0;
std::atomic<int> g_launches{0};
}  // namespace

namespace wsi {
int cuda_fail(cudaError_t e) {
  g_last_cuda_error = (int)e;
  return WS_ERR_CUDA;
}
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
}  // namespace wsi

extern "C" __attribute__((visibility("default"))) const char* ws_status_string(int status) {
  switch (status) {
    case WS_OK: return "WS_OK";
    case WS_ERR_INVALID_ARG: return "WS_ERR_INVALID_ARG: null pointer, bad size or malformed mask";
    case WS_ERR_UNSUPPORTED: return "WS_ERR_UNSUPPORTED: dtype, head_dim or mask size not compiled in";
    case WS_ERR_ALIGNMENT: return "WS_ERR_ALIGNMENT: device pointer or row pitch not 16-byte aligned";
    case WS_ERR_OUT_OF_RANGE: return "WS_ERR_OUT_OF_RANGE: rows beyond capacity or kv_visible beyond the key timeline";
    case WS_ERR_OVERLAP: return "WS_ERR_OVERLAP: source and destination ranges intersect";
    case WS_ERR_WORKSPACE: return "WS_ERR_WORKSPACE: workspace missing, misaligned or too small";
    case WS_ERR_CUDA: return "WS_ERR_CUDA: CUDA error (see ws_last_cuda_error)";
    default: return "WS_ERR_UNKNOWN";
  }
}

extern "C" __attribute__((visibility("default"))) int ws_version(void) { return WS_VERSION; }
extern "C" __attribute__((visibility("default"))) int ws_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" __attribute__((visibility("default"))) int ws_kernel_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
