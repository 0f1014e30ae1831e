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
// Nothing is barrier-synchronised: chunk k of a chain may start as soon as its chunk k-1 is stored, which a
// per-chain flag (release / acquire at GPU scope) announces; the state (72 B per particle) and the chain's
// reference energy travel through global memory, bypassing the incoherent L1.
//
// Which slots idle together matters: the slots are numbered v = (warp index on its SM) * n_sm + (rank of the SM), from
// %smid and two atomics at kernel start, so that slots that are neighbours in v -- the ones that idle together -- sit
// on different SMs, whatever order the hardware places the blocks in (with the block index as slot number a
// cooperative launch was 4 % slower than a plain one).
//
// Correct by induction on p (a position waits only for position p - M, which its slot reaches earlier in its own
// order), provided every slot is resident: the host launches the occupancy-sized grid cooperatively and falls
// back to track_kernel otherwise.  Bounded waits guard against a hang.
// The arithmetic is the fused kernel's: results are bit-identical.
#pragma once
#include "track_kernel.cuh"

#ifndef GST_CHAIN_POLL_NS
#define GST_CHAIN_POLL_NS 8192u
#endif

namespace gst {

struct ChainArgs {
  int n_chains;        // ceil(n / 32)
  int chunk_turns;     // turns per chunk
  int n_sm;            // SMs in use = gridDim.x / blocks per SM
  int* sm_scratch;     // [2 * CHAIN_MAX_SMID + 1] blocks arrived per SM, rank + 1 per SM, SMs ranked; zeroed with flag[]
  int* flag;           // [n_chains] chunks completed, zeroed before the launch
  double* E0;          // [2 n_chains] reference energy after the chain's last chunk: E0 at [c], E0lo at [n_chains + c]
  int* err;            // set to 1 when a wait times out
};

constexpr int CHAIN_MAX_SMID = 512;

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <int SPLIT, int DEPTH, int ORDER>
__global__ void __launch_bounds__(TRACK_BLOCK, TRACK_MIN_BLOCKS) track_chain_kernel(const TrackArgs a, const ChainArgs ch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // a0: stage the unique-element table and the sequence into shared memory, each when it fits
  const DevElem* tab = a.tab;
  const uint32_t* seq = a.seq;
  {
    size_t off = 0;
    if (a.use_smem_tab) {
      const int nw = a.n_unique * (int)(sizeof(DevElem) / sizeof(double));
      const double* src = reinterpret_cast<const double*>(a.tab);
      double* dst = reinterpret_cast<double*>(smem_raw);
      for (int i = threadIdx.x; i < nw; i += blockDim.x) dst[i] = src[i];
      tab = reinterpret_cast<const DevElem*>(smem_raw);
      off = (size_t)a.n_unique * sizeof(DevElem);
    }
    if (a.use_smem_seq) {
      uint32_t* sseq = reinterpret_cast<uint32_t*>(smem_raw + off);
      for (int i = threadIdx.x; i < a.n_seq; i += blockDim.x) sseq[i] = a.seq[i];
      seq = sseq;
    }
    __syncthreads();
  }
  const int lane = threadIdx.x & 31;
  const long long slots = (long long)gridDim.x * (TRACK_BLOCK / 32);
  __shared__ int s_local, s_rank;
  if (threadIdx.x == 0) {      // number the slots SM-interleaved (see the header)
    unsigned sm;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
    sm %= CHAIN_MAX_SMID;
    const int l = atomicAdd(ch.sm_scratch + sm, 1);                       // this block's index on its SM
    int rank;
    if (l == 0) {
      rank = atomicAdd(ch.sm_scratch + 2 * CHAIN_MAX_SMID, 1);
      st_release(ch.sm_scratch + CHAIN_MAX_SMID + sm, rank + 1);
    } else {
      int tries = 0;
      while ((rank = ld_acquire(ch.sm_scratch + CHAIN_MAX_SMID + sm)) == 0) {
        __nanosleep(64);
        if (++tries > (1 << 24)) { *ch.err = 1; break; }
      }
      rank -= 1;
    }
    s_local = l;
    s_rank = rank;
  }
  __syncthreads();
  if (s_rank < 0 || s_rank >= ch.n_sm || s_local * (TRACK_BLOCK / 32) >= slots / ch.n_sm) {   // not the placement assumed
    if (threadIdx.x == 0) *ch.err = 1;
    return;
  }
  const long long slot = (long long)(s_local * (TRACK_BLOCK / 32) + (threadIdx.x >> 5)) * ch.n_sm + s_rank;
  const long long n_chunks = (a.n_turns + ch.chunk_turns - 1) / ch.chunk_turns;
  const long long M = ch.n_chains;
  const long long total = n_chunks * M;
  for (long long p = slot; p < total; p += slots) {
    const long long k = p / M, c = p - k * M;             // chunk k of chain c
    if (k > 0) {                                          // chunk k-1 of this chain is stored
      // a chunk runs for milliseconds: poll with a back-off of up to GST_CHAIN_POLL_NS, so that the warps that wait
      // (320 of the 2368 slots at any time for 65 536 particles) do not take issue slots from the ones that work
      int tries = 0;
      unsigned ns = 256;
#pragma unroll 1
      while (ld_acquire(ch.flag + c) < (int)k) {
        __nanosleep(ns);
        if (ns < GST_CHAIN_POLL_NS) ns *= 2;
        if (++tries > (1 << 21)) { *ch.err = 1; return; }     // ~20 s: no chunk takes that long
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
    bool lost = false;
    typename SpinPolicy<DEPTH, SPLIT>::type spin(z);
    const long long t0 = k * ch.chunk_turns;
    const long long t1 = t0 + ch.chunk_turns < a.n_turns ? t0 + ch.chunk_turns : a.n_turns;
    uint32_t nxt = seq[0];
    for (long long turn = t0; turn < t1; ++turn) {
#pragma unroll 1
      for (int ie = 0; ie < a.n_seq; ++ie) {
        const uint32_t cur = nxt;
        nxt = seq[ie + 1 < a.n_seq ? ie + 1 : 0];
        const DevElem& e = tab[cur >> 8];
        const bool ok = element_step<SPLIT, ORDER>((int)(cur & 0xffu), z, e, pc, ref, a.G, spin);
        if (!ok) {
          lost = true;
          z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
          pcon_set(pc, 0.0, ref, a.G);
        }
      }
    }
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
    if (lane == 0) st_release(ch.flag + c, (int)k + 1);
  }
}

}  // namespace gst
