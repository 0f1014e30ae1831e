// gst_internal.h -- what gst_api.cu and gst_diag.cu share on the host side: error reporting and the device guard.
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "../../include/gst.h"

namespace gst {

extern thread_local std::string g_err;
gst_status fail(gst_status s, const char* fmt, ...);

#define CUDA_TRY(expr)                                                                           \
  do {                                                                                           \
    cudaError_t e_ = (expr);                                                                     \
    if (e_ != cudaSuccess) return gst::fail(GST_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

// Every entry point works on the device of its handle and leaves the caller's current device as it found it.
struct DeviceGuard {
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    else if (err != cudaSuccess) prev = -1;
    if (prev == dev) prev = -1;      // nothing to restore
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define GUARD_DEVICE(dev)                                                                                   \
  gst::DeviceGuard guard_(dev);                                                                             \
  if (guard_.err != cudaSuccess) return gst::fail(GST_ECUDA, "cudaSetDevice(%d): %s", (int)(dev), cudaGetErrorString(guard_.err))

}  // namespace gst
