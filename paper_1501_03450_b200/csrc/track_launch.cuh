// track_launch.cuh -- host-side launch of the tracking kernels: shared-memory plan, choice between the plain launch
// and the (chain, chunk) sequence launch, and one entry point per split so that the template instantiations of each
// split compile in their own translation unit (track_split_*.cu, built in parallel).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "track_chain_kernel.cuh"
#include "track_kernel.cuh"
#include "track_split_kernel.cuh"

namespace gst {

// what the API layer asks for: kernel arguments plus what the planner needs
struct LaunchRequest {
  TrackArgs args;
  size_t tab_bytes = 0, seq_bytes = 0;
  long long steps_per_turn = 1;
  int sms = 0;                  // SMs of the bunch's device
  bool allow_chain = false;     // GST_LAUNCH_AUTO: the planner may take the rotating launch
  bool allow_fat = true;        // not GST_LAUNCH_LEAN: small bunches take the variant with registers to spare
  bool allow_split = false;     // GST_LAUNCH_AUTO: the smallest bunches take the kernel with orbit and spin in two warps
  ChainArgs chain;              // the bunch's scratch for it (n_chains, chunk_turns, poll_limit are filled in here)
  long long poll_limit_override = 0;   // != 0: fault injection (include/gst_diag.h)
  const char* kernel = "";      // out: name of the kernel launched
};

// resources of one instantiation (gst_diag_kernel_info): what bench.py checks its flop model's capture against
struct KernelInfo { int registers = 0, local_bytes = 0, blocks_per_sm = 0; };

// The template instantiations (3 splits x 2 orders x 6 depths + 2 mid-slice orderings, each as a resident and a
// streamed kernel, plus the rotating kernels) are compiled in nine translation units that build in parallel:
// track_inst.cu with -DGST_TU_SPLIT=s -DGST_TU_GROUP=g, where group 0 = second order, depths 1-3 and the two mid-slice
// orderings, 1 = second order, depths 4-6, 2 = fourth order.  order = 2 or 4 (composition of the slice maps);
// depth >= 1: Romberg depth, 0 / -1: mid-slice PWC orderings.
#define GST_DECLARE_TU(S, G)                                                                        \
  cudaError_t launch_tu_##S##_##G(int order, int depth, LaunchRequest& rq, cudaStream_t st);         \
  cudaError_t kernel_info_tu_##S##_##G(int order, int depth, int variant, KernelInfo* out);
GST_DECLARE_TU(0, 0) GST_DECLARE_TU(0, 1) GST_DECLARE_TU(0, 2)
GST_DECLARE_TU(1, 0) GST_DECLARE_TU(1, 1) GST_DECLARE_TU(1, 2)
GST_DECLARE_TU(2, 0) GST_DECLARE_TU(2, 1) GST_DECLARE_TU(2, 2)
#undef GST_DECLARE_TU

inline int tu_group(int order, int depth) { return order == 4 ? 2 : (depth >= 4 ? 1 : 0); }
#define GST_DISPATCH_TU(FN, ...)                                                  \
  switch (split3 * 3 + tu_group(order, depth)) {                                  \
    case 0: return FN##_0_0(__VA_ARGS__);                                         \
    case 1: return FN##_0_1(__VA_ARGS__);                                         \
    case 2: return FN##_0_2(__VA_ARGS__);                                         \
    case 3: return FN##_1_0(__VA_ARGS__);                                         \
    case 4: return FN##_1_1(__VA_ARGS__);                                         \
    case 5: return FN##_1_2(__VA_ARGS__);                                         \
    case 6: return FN##_2_0(__VA_ARGS__);                                         \
    case 7: return FN##_2_1(__VA_ARGS__);                                         \
    default: return FN##_2_2(__VA_ARGS__);                                        \
  }
// split3 = SPLIT_DK / SPLIT_BK / SPLIT_MK
inline cudaError_t launch_tracking(int split3, int order, int depth, LaunchRequest& rq, cudaStream_t st) {
  GST_DISPATCH_TU(launch_tu, order, depth, rq, st)
}
// variant: 0 = track_kernel, 1 = track_chain_kernel, 2 = track_kernel (FAT), 3 = track_split_kernel
inline cudaError_t kernel_info_of(int split3, int order, int depth, int variant, KernelInfo* out) {
  GST_DISPATCH_TU(kernel_info_tu, order, depth, variant, out)
}
#undef GST_DISPATCH_TU

#ifdef GST_LAUNCH_IMPL
namespace {

// shared memory of one block (track_kernel.cuh: stage_lattice): table and sequence resident when both fit the budget
// (24 kB per block keeps 8 blocks per SM), else one record and one sequence window per warp
struct SmemPlan { size_t bytes; bool streamed; };
inline SmemPlan plan_smem(size_t tab_bytes, size_t seq_bytes, size_t budget) {
  SmemPlan p;
  p.streamed = tab_bytes + seq_bytes > budget;
  p.bytes = p.streamed ? (size_t)(TRACK_BLOCK / 32) * STREAM_BYTES_PER_WARP : tab_bytes + seq_bytes;
  return p;
}

// Does laying the (chain, chunk) work items over the warp slots pay (track_chain_kernel.cuh)?  When a plain launch
// would leave sub-partitions unevenly filled within one wave (by more than 4 %) or would need a small second wave,
// the bunch averages at least 2 warps per sub-partition (below that the static launch measured 2-5 % faster) and
// there are enough turns to cut into chunks.
inline bool chain_plan(long long n, long long n_turns, long long steps_per_turn, int slots, int sms, ChainArgs* ch) {
  const long long n_chains = (n + 31) / 32;
  const long long smsp = 4LL * sms;
  if (n_turns < 16 || n_chains < 2 * smsp || n_chains % slots == 0 || n_chains > (1LL << 30)) return false;
  if (n_chains <= slots) {
    // one wave: does the plain launch fill the sub-partitions evenly (within 4 %)?
    const long long maxw = (n_chains + smsp - 1) / smsp;
    if ((double)n_chains > 0.96 * (double)(maxw * smsp)) return false;
  } else if (2 * n_chains >= 3 * slots) {
    // one and a half waves or more: the plain launch refills the SMs block by block and its thin last wave runs
    // fast; measured (config 3, 100 turns) 131 072 / 200 000 / 262 144 particles: plain 1.67 / 1.67 / 1.73e11
    // against 1.63 / 1.65 / 1.65e11 for the sequence; 80 000 / 100 000: plain 1.34 / 1.47e11 against 1.65 / 1.64e11
    return false;
  }
  ch->n_chains = (int)n_chains;
  // a chunk of ~16k particle-element-steps (a few ms per warp) is long against the handoff and short enough to mix:
  // measured on config 3, 8 / 24 / 100 / 250 / 1000 chunks per 1000 turns give 1.56 / 1.63 / 1.65 / 1.67 / 1.67e11 steps/s
  const long long want = (16384 + steps_per_turn - 1) / std::max<long long>(1, steps_per_turn);
  ch->chunk_turns = (int)std::max<long long>(1, std::min<long long>(want, n_turns / 8));
  // Waits are bounded by progress (track_chain_kernel.cuh): a warp gives up when nothing on the chip has completed a
  // chunk for poll_limit polls of GST_CHAIN_POLL_NS each.  One chunk of S steps takes S / 8e7 s when the chip is
  // full (measured rate per warp); allow 100 times that plus 4 s, so that profilers and time-sliced GPUs do not trip it.
  const double chunk_s = (double)ch->chunk_turns * (double)steps_per_turn / 8e7;
  const double limit = (4.0 + 100.0 * chunk_s) / (GST_CHAIN_POLL_NS * 1e-9);
  ch->poll_limit = (long long)std::min(limit, 4e15);
  return true;
}

// Bunches that take the two-warp kernel: its 2 x ceil(n / 32) warps each find a sub-partition of their own.
// GST_SPLIT_MAX_WARPS_PER_SM (a build-time override for measurements) counts particle warps per SM.
#ifndef GST_SPLIT_MAX_WARPS_PER_SM
#define GST_SPLIT_MAX_WARPS_PER_SM 3
#endif
inline long long split_max_warps(int sms) { return (long long)GST_SPLIT_MAX_WARPS_PER_SM * sms; }

template <int SPLIT, int DEPTH, int ORDER>
cudaError_t launch_track(LaunchRequest& rq, cudaStream_t st) {
  TrackArgs& a = rq.args;
  const SmemPlan p = plan_smem(rq.tab_bytes, rq.seq_bytes, 24 * 1024);
  if constexpr (ORDER == 2 && DEPTH >= 1) {
    if (rq.allow_chain && !p.streamed) {   // T1c: the same arithmetic with the chains rotating over all resident warp slots
      auto ck = track_chain_kernel<SPLIT, DEPTH, ORDER>;
      int per_sm = 0;
      cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ck, TRACK_BLOCK, p.bytes);
      if (e != cudaSuccess) return e;
      // the grid never exceeds what is co-resident; when the occupancy is higher than the launch bound asks for, the
      // hardware may spread the blocks unevenly over the SMs, which the slot numbering allows for
      if (per_sm > TRACK_MIN_BLOCKS) per_sm = TRACK_MIN_BLOCKS;
      const int blocks = per_sm * rq.sms;
      ChainArgs& ca = rq.chain;
      if (blocks > 0 && chain_plan(a.n, a.n_turns, rq.steps_per_turn, blocks * (TRACK_BLOCK / 32), rq.sms, &ca)) {
        if (rq.poll_limit_override != 0) ca.poll_limit = rq.poll_limit_override;
        e = cudaMemsetAsync(ca.scratch, 0, sizeof(int) * ((size_t)ca.n_chains + CHAIN_SCRATCH_INTS), st);
        if (e != cudaSuccess) return e;
        // a cooperative launch guarantees what the hand-offs rely on: every block of the grid is resident
        void* kargs[2] = {(void*)&a, (void*)&ca};
        e = cudaLaunchCooperativeKernel((const void*)ck, dim3(blocks), dim3(TRACK_BLOCK), kargs, p.bytes, st);
        if (e == cudaSuccess) {
          rq.kernel = "track_chain_kernel";
          return cudaSuccess;
        }
        (void)cudaGetLastError();               // e.g. cudaErrorCooperativeLaunchTooLarge: take the static launch
      }
    }
  }
  if constexpr (ORDER == 2 && DEPTH >= 1) {
    // T1s: at most one warp of particles per two sub-partitions -- orbit and spin of a particle in two warps, each
    // with a sub-partition (and its FP64 pipe) to itself (track_split_kernel.cuh)
    if (rq.allow_split && !p.streamed && (a.n + 31) / 32 <= split_max_warps(rq.sms)) {
      auto sk = track_split_kernel<SPLIT, DEPTH>;
      const size_t bytes = split_ring_offset(a.n_unique, a.n_seq) + SPLIT_RING_BYTES;
      cudaError_t e = cudaFuncSetAttribute(sk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
      if (e != cudaSuccess) return e;
      sk<<<(unsigned)((a.n + 31) / 32), SPLIT_BLOCK, bytes, st>>>(a);
      rq.kernel = "track_split_kernel";
      return cudaGetLastError();
    }
  }
  // T1: one thread per particle; shared memory kept small so that 8 blocks of 64 threads stay resident
  // at most two warps per sub-partition: the variant with registers to spare (track_kernel.cuh: FAT)
  const bool fat = rq.allow_fat && !p.streamed && (a.n + 31) / 32 <= 2LL * 4 * rq.sms;
  auto kern = p.streamed ? track_kernel<SPLIT, DEPTH, ORDER, true, false>
              : fat      ? track_kernel<SPLIT, DEPTH, ORDER, false, true>
                         : track_kernel<SPLIT, DEPTH, ORDER, false, false>;
  const unsigned blocks = (unsigned)((a.n + TRACK_BLOCK - 1) / TRACK_BLOCK);
  kern<<<blocks, TRACK_BLOCK, p.bytes, st>>>(a);
  rq.kernel = fat ? "track_kernel_fat" : "track_kernel";
  return cudaGetLastError();
}

template <int SPLIT, int DEPTH, int ORDER>
cudaError_t kernel_info(int variant, KernelInfo* out) {
  const void* f = variant == 2 ? (const void*)track_kernel<SPLIT, DEPTH, ORDER, false, true>
                               : (const void*)track_kernel<SPLIT, DEPTH, ORDER, false, false>;
  int block = TRACK_BLOCK;
  if constexpr (ORDER == 2 && DEPTH >= 1) {
    if (variant == 1) f = (const void*)track_chain_kernel<SPLIT, DEPTH, ORDER>;
    if (variant == 3) { f = (const void*)track_split_kernel<SPLIT, DEPTH>; block = SPLIT_BLOCK; }
  }
  cudaFuncAttributes at;
  cudaError_t e = cudaFuncGetAttributes(&at, f);
  if (e != cudaSuccess) return e;
  out->registers = at.numRegs;
  out->local_bytes = (int)at.localSizeBytes;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&out->blocks_per_sm, f, block, 0);
}
}  // namespace
#endif  // GST_LAUNCH_IMPL

}  // namespace gst
