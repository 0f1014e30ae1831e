// track_launch.cuh -- host-side launch of the tracking kernels: shared-memory plan, choice between the plain, the
// (chain, chunk) sequence and the experimental pair launch, and one entry point per split so that the template
// instantiations of each split compile in their own translation unit (track_split_*.cu, built in parallel).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "track_chain_kernel.cuh"
#include "track_kernel.cuh"
#include "track_pair_kernel.cuh"

namespace gst {

// host-side request for the sequence launch: device arguments, what the planner needs, and whether it was taken
struct ChainLaunch {
  ChainArgs args;
  long long steps_per_turn = 1;
  bool taken = false;
};

// order = 2 or 4 (composition of the slice maps); depth >= 1: Romberg depth, 0 / -1: mid-slice PWC orderings
cudaError_t launch_split_dk(int order, int depth, const TrackArgs& a, size_t tab_bytes, size_t seq_bytes, bool pair,
                            cudaStream_t st, ChainLaunch* chain);
cudaError_t launch_split_bk(int order, int depth, const TrackArgs& a, size_t tab_bytes, size_t seq_bytes, bool pair,
                            cudaStream_t st, ChainLaunch* chain);
cudaError_t launch_split_mk(int order, int depth, const TrackArgs& a, size_t tab_bytes, size_t seq_bytes, bool pair,
                            cudaStream_t st, ChainLaunch* chain);

#ifdef GST_LAUNCH_IMPL
namespace {

// shared memory of one block: [ring + lost flags (pair kernel only)] table [sequence when it fits]
struct SmemPlan { size_t bytes; int use_smem_tab, use_smem_seq; };
SmemPlan plan_smem(size_t tab_bytes, size_t seq_bytes, size_t fixed, size_t budget) {
  SmemPlan p;
  // the table first (read at every element), then the sequence; what does not fit stays in global memory
  p.use_smem_tab = (fixed + tab_bytes <= budget) ? 1 : 0;
  const size_t with_tab = fixed + (p.use_smem_tab ? tab_bytes : 0);
  p.use_smem_seq = (with_tab + seq_bytes <= budget) ? 1 : 0;
  p.bytes = with_tab + (p.use_smem_seq ? seq_bytes : 0);
  return p;
}

// Does laying the (chain, chunk) work items over the warp slots pay (track_chain_kernel.cuh)?  When a plain launch
// would leave sub-partitions unevenly filled within one wave (by more than 4 %) or would need a small second wave,
// the bunch averages at least 2 warps per sub-partition (below that the static launch measured 2-5 % faster) and
// there are enough turns to cut into chunks.
bool chain_plan(long long n, long long n_turns, long long steps_per_turn, int slots, int sms, ChainArgs* ch) {
  const long long n_chains = (n + 31) / 32;
  const long long smsp = 4LL * sms;
  if (n_turns < 16 || n_chains < 2 * smsp || n_chains % slots == 0) return false;
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
  return true;
}

template <int SPLIT, int DEPTH, int ORDER>
cudaError_t launch_track(TrackArgs a, size_t tab_bytes, size_t seq_bytes, bool pair, cudaStream_t st,
                         ChainLaunch* chain = nullptr) {
  if constexpr (ORDER == 2 && DEPTH >= 1) {   // the experimental pair kernel: second-order maps, edge scheme only
  if (pair) {
    // T1p: two threads per particle.  Shared memory per block is budgeted so that MIN_BLOCKS blocks stay
    // resident per SM (227 kB usable, 1 kB reserved per block).
    using Cfg = PairCfg<DEPTH>;
    auto kern = track_pair_kernel<SPLIT, DEPTH>;
    const size_t fixed = (size_t)Cfg::PAIRS * (PAIR_RING_BYTES + 32);
    const size_t budget = (size_t)(227 * 1024) / Cfg::MIN_BLOCKS - 1024;
    SmemPlan p = plan_smem(tab_bytes, seq_bytes, fixed, budget);

    a.use_smem_seq = p.use_smem_seq;
  a.use_smem_tab = p.use_smem_tab;
    a.use_smem_tab = p.use_smem_tab;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
    if (e != cudaSuccess) return e;
    // ask for just enough shared memory for MIN_BLOCKS blocks; the rest of the 228 kB stays L1
    int carve = (int)(((p.bytes + 1024) * Cfg::MIN_BLOCKS * 100 + 228 * 1024 - 1) / (228 * 1024));
    if (carve > 100) carve = 100;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
    if (e != cudaSuccess) return e;
    const long long per_block = 32LL * Cfg::PAIRS;
    unsigned blocks = (unsigned)((a.n + per_block - 1) / per_block);
    kern<<<blocks, Cfg::THREADS, p.bytes, st>>>(a);
    return cudaGetLastError();
  }
  }
  SmemPlan p = plan_smem(tab_bytes, seq_bytes, 0, 24 * 1024);
  a.use_smem_seq = p.use_smem_seq;
  a.use_smem_tab = p.use_smem_tab;
  if constexpr (ORDER == 2 && DEPTH >= 1) {
    if (chain) {   // T1c: the same kernel with the chains rotating over all resident warp slots
      auto ck = track_chain_kernel<SPLIT, DEPTH, ORDER>;
      int dev = 0, sms = 0, per_sm = 0;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      if (p.bytes > 48 * 1024) cudaFuncSetAttribute(ck, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
      cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ck, TRACK_BLOCK, p.bytes);
      if (e != cudaSuccess) return e;
      if (per_sm > TRACK_MIN_BLOCKS) per_sm = TRACK_MIN_BLOCKS;
      const int blocks = per_sm * sms;
      ChainArgs& ca = chain->args;
      if (chain_plan(a.n, a.n_turns, chain->steps_per_turn, blocks * (TRACK_BLOCK / 32), sms, &ca)) {
        ca.n_sm = sms;
        e = cudaMemsetAsync(ca.sm_scratch, 0, sizeof(int) * (ca.n_chains + 2 * CHAIN_MAX_SMID + 1), st);
        if (e != cudaSuccess) return e;
        // a cooperative launch guarantees what the hand-offs rely on: every block of the grid is resident
        void* kargs[2] = {(void*)&a, (void*)&ca};
        e = cudaLaunchCooperativeKernel((const void*)ck, dim3(blocks), dim3(TRACK_BLOCK), kargs, p.bytes, st);
        if (e == cudaSuccess) {
          chain->taken = true;
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
  unsigned blocks = (unsigned)((a.n + TRACK_BLOCK - 1) / TRACK_BLOCK);
  kern<<<blocks, TRACK_BLOCK, p.bytes, st>>>(a);
  return cudaGetLastError();
}

template <int SPLIT, int ORDER>
cudaError_t launch_track_depth(int depth, const TrackArgs& a, size_t tb, size_t sb, bool pair, cudaStream_t st,
                               ChainLaunch* chain) {
  if (ORDER == 2 && depth == 0) return launch_track<SPLIT, 0, 2>(a, tb, sb, false, st);
  if (ORDER == 2 && depth == -1) return launch_track<SPLIT, -1, 2>(a, tb, sb, false, st);
  switch (depth) {
    case 1: return launch_track<SPLIT, 1, ORDER>(a, tb, sb, pair, st, chain);
    case 2: return launch_track<SPLIT, 2, ORDER>(a, tb, sb, pair, st, chain);
    case 3: return launch_track<SPLIT, 3, ORDER>(a, tb, sb, pair, st, chain);
    case 4: return launch_track<SPLIT, 4, ORDER>(a, tb, sb, pair, st, chain);
    case 5: return launch_track<SPLIT, 5, ORDER>(a, tb, sb, pair, st, chain);
    default: return launch_track<SPLIT, 6, ORDER>(a, tb, sb, pair, st, chain);
  }
}


template <int SPLIT>
cudaError_t launch_split(int order, int depth, const TrackArgs& a, size_t tb, size_t sb, bool pair, cudaStream_t st,
                         ChainLaunch* chain) {
  if (order == 4) return launch_track_depth<SPLIT, 4>(depth, a, tb, sb, pair, st, chain);
  return launch_track_depth<SPLIT, 2>(depth, a, tb, sb, pair, st, chain);
}

}  // namespace
#endif  // GST_LAUNCH_IMPL

}  // namespace gst
