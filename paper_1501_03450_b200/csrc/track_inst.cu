// track_inst.cu -- one translation unit of tracking-kernel instantiations: compiled nine times with
// -DGST_TU_SPLIT=0|1|2 (drift-, bend-, matrix-kick) and -DGST_TU_GROUP=0|1|2 (see track_launch.cuh).
// -DGST_ONLY_DEPTH=d (development builds that compile in seconds) keeps the kernels of Romberg depth d alone (both
// orders, no mid-slice orderings); every other request fails with cudaErrorNotSupported.
#define GST_LAUNCH_IMPL
#include "track_launch.cuh"

#define GST_CAT4_(a, b, c) a##_##b##_##c
#define GST_CAT4(a, b, c) GST_CAT4_(a, b, c)

namespace gst {

#ifdef GST_ONLY_DEPTH
#define GST_CASE(D, O) case D: if (D != GST_ONLY_DEPTH) return cudaErrorNotSupported; else
#else
#define GST_CASE(D, O) case D:
#endif

cudaError_t GST_CAT4(launch_tu, GST_TU_SPLIT, GST_TU_GROUP)(int order, int depth, LaunchRequest& rq, cudaStream_t st) {
  constexpr int S = GST_TU_SPLIT;
  (void)order;
  switch (depth) {
#if GST_TU_GROUP == 0
#ifndef GST_ONLY_DEPTH
    case 0: return launch_track<S, 0, 2>(rq, st);
    case -1: return launch_track<S, -1, 2>(rq, st);
#endif
#if !defined(GST_ONLY_DEPTH) || GST_ONLY_DEPTH <= 3
    GST_CASE(1, 2) return launch_track<S, 1, 2>(rq, st);
    GST_CASE(2, 2) return launch_track<S, 2, 2>(rq, st);
    GST_CASE(3, 2) return launch_track<S, 3, 2>(rq, st);
#endif
#elif GST_TU_GROUP == 1
#if !defined(GST_ONLY_DEPTH) || GST_ONLY_DEPTH >= 4
    GST_CASE(4, 2) return launch_track<S, 4, 2>(rq, st);
    GST_CASE(5, 2) return launch_track<S, 5, 2>(rq, st);
    GST_CASE(6, 2) return launch_track<S, 6, 2>(rq, st);
#endif
#elif defined(GST_ONLY_DEPTH)
    case GST_ONLY_DEPTH: return launch_track<S, GST_ONLY_DEPTH, 4>(rq, st);
#else
    case 1: return launch_track<S, 1, 4>(rq, st);
    case 2: return launch_track<S, 2, 4>(rq, st);
    case 3: return launch_track<S, 3, 4>(rq, st);
    case 4: return launch_track<S, 4, 4>(rq, st);
    case 5: return launch_track<S, 5, 4>(rq, st);
    case 6: return launch_track<S, 6, 4>(rq, st);
#endif
    default: return cudaErrorNotSupported;
  }
}

cudaError_t GST_CAT4(kernel_info_tu, GST_TU_SPLIT, GST_TU_GROUP)(int order, int depth, int variant, KernelInfo* out) {
  constexpr int S = GST_TU_SPLIT;
  (void)order;
  switch (depth) {
#if GST_TU_GROUP == 0
#ifndef GST_ONLY_DEPTH
    case 0: return kernel_info<S, 0, 2>(variant, out);
    case -1: return kernel_info<S, -1, 2>(variant, out);
#endif
#if !defined(GST_ONLY_DEPTH) || GST_ONLY_DEPTH <= 3
    GST_CASE(1, 2) return kernel_info<S, 1, 2>(variant, out);
    GST_CASE(2, 2) return kernel_info<S, 2, 2>(variant, out);
    GST_CASE(3, 2) return kernel_info<S, 3, 2>(variant, out);
#endif
#elif GST_TU_GROUP == 1
#if !defined(GST_ONLY_DEPTH) || GST_ONLY_DEPTH >= 4
    GST_CASE(4, 2) return kernel_info<S, 4, 2>(variant, out);
    GST_CASE(5, 2) return kernel_info<S, 5, 2>(variant, out);
    GST_CASE(6, 2) return kernel_info<S, 6, 2>(variant, out);
#endif
#elif defined(GST_ONLY_DEPTH)
    case GST_ONLY_DEPTH: return kernel_info<S, GST_ONLY_DEPTH, 4>(variant, out);
#else
    case 1: return kernel_info<S, 1, 4>(variant, out);
    case 2: return kernel_info<S, 2, 4>(variant, out);
    case 3: return kernel_info<S, 3, 4>(variant, out);
    case 4: return kernel_info<S, 4, 4>(variant, out);
    case 5: return kernel_info<S, 5, 4>(variant, out);
    case 6: return kernel_info<S, 6, 4>(variant, out);
#endif
    default: return cudaErrorNotSupported;
  }
}

}  // namespace gst
