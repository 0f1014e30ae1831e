// track_split_mk.cu -- instantiations of the tracking kernels for one split (see track_launch.cuh)
#define GST_LAUNCH_IMPL
#include "track_launch.cuh"

namespace gst {
cudaError_t launch_split_mk(int order, int depth, const TrackArgs& a, size_t tab_bytes, size_t seq_bytes, bool pair,
                            cudaStream_t st, ChainLaunch* chain) {
  return launch_split<SPLIT_MK>(order, depth, a, tab_bytes, seq_bytes, pair, st, chain);
}
}  // namespace gst
