// track_split_mk.cu -- instantiations of the tracking kernels for one split (see track_launch.cuh)
#define GST_LAUNCH_IMPL
#include "track_launch.cuh"

namespace gst {
cudaError_t launch_split_mk(int order, int depth, LaunchRequest& rq, cudaStream_t st) {
  return launch_split<SPLIT_MK>(order, depth, rq, st);
}
cudaError_t kernel_info_mk(int order, int depth, bool chain, KernelInfo* out) {
  return kernel_info_split<SPLIT_MK>(order, depth, chain, out);
}
}  // namespace gst
