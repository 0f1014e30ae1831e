// track_chain_kernel.cuh -- T1c: the fused tracking kernel with the bunch ROTATING over the warp slots of the chip.
//
// Why: a bunch of 65 536 particles is 2048 warps ("chains" of 32 particles) on 592 SM sub-partitions: 272 of
// them hold 4 warps and 320 hold 3.  A sub-partition with 4 warps is saturated (profiles/r01_notes.md), so in
// track_kernel.cuh the 3-warp ones finish after 77 % of the time and idle: 13 % of the chip's FP64 cycles.  A
// bunch of 262 144 particles is 3.46 WAVES of blocks, and the last wave leaves half the chip empty.
// Here the grid is exactly the S = 4 x 592 warp slots the chip holds, the turns are cut into chunks, and the
// work items (chain c, chunk k) are laid out in one sequence  p = k * M + c  (M chains): slot v takes the
// positions p = v, v + S, v + 2S, ...  Consecutive chunks of a chain are M positions apart, so
//   M > S : every slot is busy all the time and a chain rests in global memory between its chunks -- no waves;
//   M < S : in every round S - M slots find that their chain's previous chunk is still being computed and
//           wait; because S is not a multiple of M these idle slots wander over the chip, so every
//           sub-partition carries the same load over the launch.
// Nothing but the start is barrier-synchronised: chunk k of a chain may start as soon as its chunk k-1 is stored,
// which a per-chain flag (release / acquire at GPU scope) announces; the state (72 B per particle) and the chain's
// reference energy travel through global memory, bypassing the incoherent L1.
//
// Which slots idle together matters: neighbours in the slot number v -- the ones that idle together -- must sit on
// different SMs, whatever order the hardware places the blocks in (with the block index as slot number a cooperative
// launch was 4 % slower than a plain one).  Every block therefore registers on its SM (%smid: its index l among the
// blocks there, the SM's rank by first arrival), all blocks meet once at a start barrier (the launch is cooperative,
// so they are co-resident), and then each computes its number from the final per-SM counts:
//   v = 2 * #{blocks with index < l} + w * n_l + #{SMs that hold more than l blocks and rank below this one's},
// w = warp in the block, n_l = SMs holding more than l blocks.  This is a bijection onto 0..S-1 for ANY distribution
// of the blocks over the SMs (a cooperative launch guarantees co-residency, not an even spread), and SM-interleaved.
//
// Correct by induction on p (a position waits only for position p - M, which its slot reaches earlier in its own
// order), provided every slot is resident: the host launches the grid cooperatively and falls back to track_kernel
// when that is refused.  Waits are bounded by PROGRESS: a waiting warp gives up when no chunk anywhere on the chip
// has completed for `poll_limit` polls (scaled by the host with the length of a chunk), sets the bunch's error word
// and leaves; everybody else follows.  The arithmetic is the fused kernel's: results are bit-identical.
#pragma once
#include "track_kernel.cuh"

#ifndef GST_CHAIN_POLL_NS
#define GST_CHAIN_POLL_NS 8192u
#endif

namespace gst {

constexpr int CHAIN_MAX_SMID = 512;
// layout of the per-bunch int scratch, zeroed (together with the chain flags behind it) before every rotating launch
constexpr int CHAIN_COUNT = 0;                        // [CHAIN_MAX_SMID] blocks registered per SM
constexpr int CHAIN_RANK = CHAIN_MAX_SMID;            // [CHAIN_MAX_SMID] rank + 1 of the SM by first arrival
constexpr int CHAIN_NRANKED = 2 * CHAIN_MAX_SMID;     // SMs ranked so far
constexpr int CHAIN_ARRIVED = 2 * CHAIN_MAX_SMID + 1; // blocks at the start barrier
constexpr int CHAIN_PROGRESS = 2 * CHAIN_MAX_SMID + 2;// chunks completed, all chains
constexpr int CHAIN_SCRATCH_INTS = 2 * CHAIN_MAX_SMID + 4;

struct ChainArgs {
  int n_chains;          // ceil(n / 32)
  int chunk_turns;       // turns per chunk
  int* scratch;          // [CHAIN_SCRATCH_INTS], see above
  int* flag;             // [n_chains] chunks completed per chain
  double* E0;            // [2 n_chains] reference energy after the chain's last chunk: E0 at [c], E0lo at [n_chains + c]
  int* err;              // the bunch's error word (sticky until the host reports it)
  long long poll_limit;  // > 0: give up after this many polls WITHOUT PROGRESS anywhere; < 0: after -poll_limit polls
                         // whatever happens elsewhere (fault injection, include/gst_diag.h)
};

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int ld_relaxed(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Number this block's first warp slot (see the header).  Returns -1 when the start barrier timed out.
__device__ __forceinline__ long long chain_slot_of_block(const ChainArgs& ch, int warps_per_block) {
  __shared__ int s_l, s_rank, s_part[3];
  int* sc = ch.scratch;
  if (threadIdx.x == 0) {
    unsigned sm;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
    sm %= CHAIN_MAX_SMID;
    const int l = atomicAdd(sc + CHAIN_COUNT + sm, 1);                    // this block's index on its SM
    if (l == 0) st_release(sc + CHAIN_RANK + sm, atomicAdd(sc + CHAIN_NRANKED, 1) + 1);
    __threadfence();
    atomicAdd(sc + CHAIN_ARRIVED, 1);
    int tries = 0;
    bool ok = true;
    while (ld_acquire(sc + CHAIN_ARRIVED) < (int)gridDim.x) {             // start barrier: the counts are final after it
      __nanosleep(128);
      if (++tries > (1 << 22) || ld_relaxed(ch.err) != 0) { ok = false; break; }
    }
    s_l = ok ? l : -1;
    s_rank = ok ? ld_acquire(sc + CHAIN_RANK + sm) - 1 : -1;
    s_part[0] = s_part[1] = s_part[2] = 0;
  }
  __syncthreads();
  const int l = s_l, rank = s_rank;
  if (l < 0 || rank < 0) return -1;
  // blocks with a smaller index, SMs on this level, SMs on this level ranked below this one: summed over the SM ids
  int below = 0, level = 0, before = 0;
  for (int s = threadIdx.x; s < CHAIN_MAX_SMID; s += blockDim.x) {
    const int c = ld_relaxed(sc + CHAIN_COUNT + s);
    if (c == 0) continue;
    below += c < l ? c : l;
    if (c > l) {
      ++level;
      if (ld_relaxed(sc + CHAIN_RANK + s) - 1 < rank) ++before;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    below += __shfl_down_sync(0xffffffffu, below, o);
    level += __shfl_down_sync(0xffffffffu, level, o);
    before += __shfl_down_sync(0xffffffffu, before, o);
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&s_part[0], below);
    atomicAdd(&s_part[1], level);
    atomicAdd(&s_part[2], before);
  }
  __syncthreads();
  // warp w of this block: slot = warps_per_block * below + w * level + before
  return ((long long)s_part[1] << 32) | (unsigned)(warps_per_block * s_part[0] + s_part[2]);
}

template <int SPLIT, int DEPTH, int ORDER>
__global__ void __launch_bounds__(TRACK_BLOCK, TRACK_MIN_BLOCKS) track_chain_kernel(const TrackArgs a, const ChainArgs ch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  stage_lattice<false>(a, smem_raw);                     // the planner takes this kernel only when the lattice is resident
  if (*a.err != 0) return;                               // an earlier launch on this bunch failed: leave everything (gst.h)
  const int lane = threadIdx.x & 31;
  const long long slots = (long long)gridDim.x * (TRACK_BLOCK / 32);
  const long long packed = chain_slot_of_block(ch, TRACK_BLOCK / 32);
  if (packed < 0) {
    if (threadIdx.x == 0) atomicExch(ch.err, 1);
    return;
  }
  const long long slot = (long long)(unsigned)(packed & 0xffffffffLL) + (long long)(threadIdx.x >> 5) * (packed >> 32);
  const long long n_chunks = (a.n_turns + ch.chunk_turns - 1) / ch.chunk_turns;
  const long long M = ch.n_chains;
  const long long total = n_chunks * M;
  int* progress = ch.scratch + CHAIN_PROGRESS;
  for (long long p = slot; p < total; p += slots) {
    const long long k = p / M, c = p - k * M;             // chunk k of chain c
    if (k > 0) {                                          // chunk k-1 of this chain is stored
      // a chunk runs for milliseconds: poll with a back-off of up to GST_CHAIN_POLL_NS, so that the warps that wait
      // (320 of the 2368 slots at any time for 65 536 particles) do not take issue slots from the ones that work
      long long polls = 0, idle = 0;
      int seen = 0;
      unsigned ns = 256;
#pragma unroll 1
      while (ld_acquire(ch.flag + c) < (int)k) {
        __nanosleep(ns);
        if (ns < GST_CHAIN_POLL_NS) ns *= 2;
        ++polls;
        if ((polls & 15) == 0 || ch.poll_limit < 0) {     // every 16th poll: has anything on the chip moved?
          const int now = ld_relaxed(progress);
          idle = now != seen ? 0 : idle + 16;
          seen = now;
          const bool out_of_time = ch.poll_limit > 0 ? idle > ch.poll_limit : polls > -ch.poll_limit;
          if (out_of_time || ld_relaxed(ch.err) != 0) {
            atomicExch(ch.err, 1);
            return;
          }
        }
      }
    }
    const long long j = c * 32 + lane;
    const bool valid = j < a.n && !__ldcg(a.lost + j);
    State z;
    z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
    z.Sx = 0.0; z.Sy = 1.0; z.Ss = 0.0;
    if (valid) {
      z.X = __ldcg(a.p[0] + j); z.Px = __ldcg(a.p[1] + j); z.Y = __ldcg(a.p[2] + j); z.Py = __ldcg(a.p[3] + j);
      z.T = __ldcg(a.p[4] + j); z.Pt = __ldcg(a.p[5] + j);
      z.Sx = __ldcg(a.p[6] + j); z.Sy = __ldcg(a.p[7] + j); z.Ss = __ldcg(a.p[8] + j);
    }
    Ref ref;
    ref_set(ref, k == 0 ? a.E0 : __ldcg(ch.E0 + c), a.mass);
    ref.E0lo = k == 0 ? a.E0lo : __ldcg(ch.E0 + ch.n_chains + c);
    PCon pc;
    pcon_set(pc, z.Pt, ref, a.G);
    typename SpinPolicy<DEPTH, SPLIT, false>::type spin(z);
    const long long t0 = k * ch.chunk_turns;
    const long long t1 = t0 + ch.chunk_turns < a.n_turns ? t0 + ch.chunk_turns : a.n_turns;
    const bool lost = track_turns<SPLIT, ORDER, false>(z, ref, pc, spin, t0, t1, a, smem_raw);
    if (valid) {
      if (lost) {
        a.lost[j] = 1;
      } else {
        __stcg(a.p[0] + j, z.X); __stcg(a.p[1] + j, z.Px); __stcg(a.p[2] + j, z.Y); __stcg(a.p[3] + j, z.Py);
        __stcg(a.p[4] + j, z.T); __stcg(a.p[5] + j, z.Pt);
        __stcg(a.p[6] + j, z.Sx); __stcg(a.p[7] + j, z.Sy); __stcg(a.p[8] + j, z.Ss);
      }
    }
    if (lane == 0) {
      __stcg(ch.E0 + c, ref.E0);
      __stcg(ch.E0 + ch.n_chains + c, ref.E0lo);
    }
    __threadfence();
    __syncwarp();
    if (lane == 0) {
      st_release(ch.flag + c, (int)k + 1);
      atomicAdd(progress, 1);
    }
  }
}

}  // namespace gst
