// track_launch.cuh -- host-side launch of the tracking kernels: shared-memory plan, choice between the plain launch
// and the (chain, chunk) sequence launch, and one entry point per split so that the template instantiations of each
// split compile in their own translation unit (track_split_*.cu, built in parallel).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "track_chain_kernel.cuh"
#include "track_kernel.cuh"

namespace gst {

// what the API layer asks for: kernel arguments plus what the planner needs
struct LaunchRequest {
  TrackArgs args;
  size_t tab_bytes = 0, seq_bytes = 0;
  long long steps_per_turn = 1;
  int sms = 0;                  // SMs of the bunch's device
  bool allow_chain = false;     // GST_LAUNCH_AUTO: the planner may take the rotating launch
  ChainArgs chain;              // the bunch's scratch for it (n_chains, chunk_turns, poll_limit are filled in here)
  long long poll_limit_override = 0;   // != 0: fault injection (include/gst_diag.h)
  const char* kernel = "";      // out: name of the kernel launched
};

// order = 2 or 4 (composition of the slice maps); depth >= 1: Romberg depth, 0 / -1: mid-slice PWC orderings
cudaError_t launch_split_dk(int order, int depth, LaunchRequest& rq, cudaStream_t st);
cudaError_t launch_split_bk(int order, int depth, LaunchRequest& rq, cudaStream_t st);
cudaError_t launch_split_mk(int order, int depth, LaunchRequest& rq, cudaStream_t st);

// resources of one instantiation (gst_diag_kernel_info): what bench.py checks its flop model's capture against
struct KernelInfo { int registers = 0, local_bytes = 0, blocks_per_sm = 0; };
cudaError_t kernel_info_dk(int order, int depth, bool chain, KernelInfo* out);
cudaError_t kernel_info_bk(int order, int depth, bool chain, KernelInfo* out);
cudaError_t kernel_info_mk(int order, int depth, bool chain, KernelInfo* out);

#ifdef GST_LAUNCH_IMPL
namespace {

// shared memory of one block: table [sequence when it fits]
struct SmemPlan { size_t bytes; int use_smem_tab, use_smem_seq; };
inline SmemPlan plan_smem(size_t tab_bytes, size_t seq_bytes, size_t budget) {
  SmemPlan p;
  // the table first (read at every element), then the sequence; what does not fit stays in global memory
  p.use_smem_tab = (tab_bytes <= budget) ? 1 : 0;
  const size_t with_tab = p.use_smem_tab ? tab_bytes : 0;
  p.use_smem_seq = (with_tab + seq_bytes <= budget) ? 1 : 0;
  p.bytes = with_tab + (p.use_smem_seq ? seq_bytes : 0);
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

template <int SPLIT, int DEPTH, int ORDER>
cudaError_t launch_track(LaunchRequest& rq, cudaStream_t st) {
  TrackArgs& a = rq.args;
  const SmemPlan p = plan_smem(rq.tab_bytes, rq.seq_bytes, 24 * 1024);
  a.use_smem_seq = p.use_smem_seq;
  a.use_smem_tab = p.use_smem_tab;
  if constexpr (ORDER == 2 && DEPTH >= 1) {
    if (rq.allow_chain) {   // T1c: the same arithmetic with the chains rotating over all resident warp slots
      auto ck = track_chain_kernel<SPLIT, DEPTH, ORDER>;
      int per_sm = 0;
      if (p.bytes > 48 * 1024) cudaFuncSetAttribute(ck, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
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
  // T1: one thread per particle; shared memory kept small so that 8 blocks of 64 threads stay resident
  auto kern = track_kernel<SPLIT, DEPTH, ORDER>;
  if (p.bytes > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
    if (e != cudaSuccess) return e;
  }
  const unsigned blocks = (unsigned)((a.n + TRACK_BLOCK - 1) / TRACK_BLOCK);
  kern<<<blocks, TRACK_BLOCK, p.bytes, st>>>(a);
  rq.kernel = "track_kernel";
  return cudaGetLastError();
}

// -DGST_ONLY_DEPTH=d builds the edge-scheme kernels of Romberg depth d alone (second order; development builds that
// compile in seconds): every other request fails with cudaErrorNotSupported.
template <int SPLIT, int ORDER>
cudaError_t launch_track_depth(int depth, LaunchRequest& rq, cudaStream_t st) {
#ifdef GST_ONLY_DEPTH
  if constexpr (ORDER == 2) {
    if (depth == GST_ONLY_DEPTH) return launch_track<SPLIT, GST_ONLY_DEPTH, 2>(rq, st);
  }
  return cudaErrorNotSupported;
#else
  if (ORDER == 2 && depth == 0) return launch_track<SPLIT, 0, 2>(rq, st);
  if (ORDER == 2 && depth == -1) return launch_track<SPLIT, -1, 2>(rq, st);
  switch (depth) {
    case 1: return launch_track<SPLIT, 1, ORDER>(rq, st);
    case 2: return launch_track<SPLIT, 2, ORDER>(rq, st);
    case 3: return launch_track<SPLIT, 3, ORDER>(rq, st);
    case 4: return launch_track<SPLIT, 4, ORDER>(rq, st);
    case 5: return launch_track<SPLIT, 5, ORDER>(rq, st);
    default: return launch_track<SPLIT, 6, ORDER>(rq, st);
  }
#endif
}

template <int SPLIT, int DEPTH, int ORDER>
cudaError_t kernel_info(bool chain, KernelInfo* out) {
  const void* f = (const void*)track_kernel<SPLIT, DEPTH, ORDER>;
  if constexpr (ORDER == 2 && DEPTH >= 1) {
    if (chain) f = (const void*)track_chain_kernel<SPLIT, DEPTH, ORDER>;
  }
  cudaFuncAttributes at;
  cudaError_t e = cudaFuncGetAttributes(&at, f);
  if (e != cudaSuccess) return e;
  out->registers = at.numRegs;
  out->local_bytes = (int)at.localSizeBytes;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&out->blocks_per_sm, f, TRACK_BLOCK, 0);
}
template <int SPLIT>
cudaError_t kernel_info_split(int order, int depth, bool chain, KernelInfo* out) {
#ifdef GST_ONLY_DEPTH
  if (order == 2 && depth == GST_ONLY_DEPTH) return kernel_info<SPLIT, GST_ONLY_DEPTH, 2>(chain, out);
  return cudaErrorNotSupported;
#else
#define GST_KI(D)                                                          \
  case D: return order == 4 ? kernel_info<SPLIT, D, 4>(chain, out) : kernel_info<SPLIT, D, 2>(chain, out);
  switch (depth) {
    GST_KI(1) GST_KI(2) GST_KI(3) GST_KI(4) GST_KI(5)
    default: return order == 4 ? kernel_info<SPLIT, 6, 4>(chain, out) : kernel_info<SPLIT, 6, 2>(chain, out);
  }
#undef GST_KI
#endif
}

template <int SPLIT>
cudaError_t launch_split(int order, int depth, LaunchRequest& rq, cudaStream_t st) {
  if (order == 4) return launch_track_depth<SPLIT, 4>(depth, rq, st);
  return launch_track_depth<SPLIT, 2>(depth, rq, st);
}

}  // namespace
#endif  // GST_LAUNCH_IMPL

}  // namespace gst
