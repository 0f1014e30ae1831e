// track_pair_kernel.cuh -- T1p: EXPERIMENTAL variant of the tracking kernel with TWO threads per particle
// (sm_100a, fp64).  Selected with gst_set_kernel_variant(GST_KERNEL_PAIR); the default is the fused
// one-thread-per-particle kernel of track_kernel.cuh, which is faster on every workload measured so far
// (profiles/r01_notes.md, "pair kernel").
//
// Idea: BASELINE's headline bunch has 65 536 particles = 2048 warps on 592 SM sub-partitions, i.e. 3 or 4
// warps of one long dependent fp64 chain each.  The spin motion never feeds back into the orbit
// (6a)(6b), so a particle can be split into a pipeline of two threads:
//
//   orbit thread : 6-D state, element maps, w*ds*Omega at every slice edge and its quaternion (a2-a9, a10a)
//   spin thread  : DEPTH level products, Romberg, S <- Q S Q*, snakes                         (a10b-a12)
//
// Lane l of the block's "orbit warp" and lane l of its "spin warp" serve the same particle; the edge
// quaternions (4 doubles) travel through a small shared-memory ring (PAIR_NST stages of PAIR_CH edges,
// 1 kB per edge) guarded by hardware named barriers (bar.arrive / bar.sync with a count of 64).  Both
// warps walk the same element sequence, so the consumer knows how many edges each element delivers;
// nothing else is communicated.  This doubles the warps (6.9 per sub-partition, evenly spread) at
// 72 registers each.
//
// What was measured (B200, config 3): the variant executes 1.6x the warp instructions of the fused
// kernel (ring addressing, barriers, rolled loops) and its warps spend a quarter of their time in
// bar.sync because 15 kB of shared memory per pair buffers less than one element (8 edges); 1.0e11
// particle-element-steps/s against 1.29e11 fused.  Kept because it is correct (bit-identical results,
// tested) and the obvious next step if shared memory per SM grows.
//
// The arithmetic is the same code as the fused kernel (same steppers, same quaternion routines).
#pragma once
#include "track_kernel.cuh"

namespace gst {

constexpr int PAIR_CH = 4;    // edges per ring stage
constexpr int PAIR_NST = 2;   // ring stages
constexpr int PAIR_SLOTS = PAIR_CH * PAIR_NST;
constexpr int PAIR_EDGE_DOUBLES = 4 * 32;                             // one edge of one warp pair
constexpr int PAIR_RING_BYTES = PAIR_SLOTS * PAIR_EDGE_DOUBLES * 8;   // 8192 B per pair

// Named barriers are a per-SM resource (64), and the ids must be immediates (with an id in a register
// ptxas reserves all 16 per block).  A block is ONE warp pair (64 threads) and owns barriers 0..3, so 14
// blocks fit per SM; code that runs on both pairs of a bigger block would need the pair index at compile
// time, i.e. two copies of every loop in the instruction cache (measured: 1.5x slower).
//   full[st]  = 2 st       (producer arrives, consumer waits)     empty[st] = 2 st + 1  (the reverse)
// Barrier 0 is also __syncthreads(): it is used that way only before the ring starts and after it has
// drained, when full[0] has no pending arrival.
template <int ID> __device__ __forceinline__ void bar_sync_imm() { asm volatile("bar.sync %0, 64;" ::"n"(ID) : "memory"); }
template <int ID> __device__ __forceinline__ void bar_arrive_imm() { asm volatile("bar.arrive %0, 64;" ::"n"(ID) : "memory"); }

// One end of the ring.  `slot` is uniform across the warp (all lanes are at the same edge).
struct Chan {
  double* base;   // the ring, already offset by the lane
  int slot;       // next slot to write / read, 0..PAIR_SLOTS-1
  static_assert(PAIR_NST == 2, "two stages: the stage is one bit of the slot");
  __device__ __forceinline__ void wait_full(int st) { if (st) bar_sync_imm<2>(); else bar_sync_imm<0>(); }
  __device__ __forceinline__ void signal_full(int st) { if (st) bar_arrive_imm<2>(); else bar_arrive_imm<0>(); }
  __device__ __forceinline__ void wait_empty(int st) { if (st) bar_sync_imm<3>(); else bar_sync_imm<1>(); }
  __device__ __forceinline__ void signal_empty(int st) { if (st) bar_arrive_imm<3>(); else bar_arrive_imm<1>(); }
};

// ---- producer side (orbit thread) ------------------------------------------------------------
struct PushSpin {
  Chan& c;
  __device__ __forceinline__ explicit PushSpin(Chan& c_) : c(c_) {}
  __device__ __forceinline__ void push(const Quat& q) {
    const int st = c.slot / PAIR_CH, k = c.slot % PAIR_CH;
    if (k == 0) c.wait_empty(st);                  // the consumer has released this stage
    double* p = c.base + c.slot * PAIR_EDGE_DOUBLES;
    p[0] = q.w; p[32] = q.x; p[64] = q.y; p[96] = q.s;
    if (k == PAIR_CH - 1) c.signal_full(st);
    c.slot = (c.slot + 1) % PAIR_SLOTS;
  }
  // after the last element: hand over a partly filled stage
  __device__ __forceinline__ void flush() {
    if (c.slot % PAIR_CH != 0) c.signal_full(c.slot / PAIR_CH);
  }
  template <class Stepper>
  __device__ __forceinline__ void run(Stepper& s, int N, double ds) {
    const double hds = 0.5 * ds;
    double wx, wy, ws;
    s.omega(hds, wx, wy, ws);                       // edge 0, half weight
    Quat q = quat_from_rotvec(wx, wy, ws);
#pragma unroll 1
    for (int i = 1; i <= N; ++i) {
      s.advance();                                  // slice i is independent of the store of edge i-1
      push(q);
      s.omega(i == N ? hds : ds, wx, wy, ws);
      q = quat_from_rotvec(wx, wy, ws);
    }
    push(q);
  }
  __device__ __forceinline__ void thin(double wx, double wy, double ws) { push(quat_from_rotvec(wx, wy, ws)); }
  __device__ __forceinline__ void snake(const Quat&) {}
};

// ---- consumer side (spin thread) -------------------------------------------------------------
struct PopSpin {
  Chan& c;
  __device__ __forceinline__ explicit PopSpin(Chan& c_) : c(c_) {}
  __device__ __forceinline__ void start() {           // every stage starts empty
    c.signal_empty(0);
    c.signal_empty(1);
  }
  __device__ __forceinline__ Quat pop() {
    const int st = c.slot / PAIR_CH, k = c.slot % PAIR_CH;
    if (k == 0) c.wait_full(st);                   // the producer has filled this stage
    const double* p = c.base + c.slot * PAIR_EDGE_DOUBLES;
    Quat q{p[0], p[32], p[64], p[96]};
    if (k == PAIR_CH - 1) c.signal_empty(st);      // stage released (the loads above are ordered before it)
    c.slot = (c.slot + 1) % PAIR_SLOTS;
    return q;
  }
  // the N+1 edges of a thick element.  Edge i belongs to level l when 2^l | i (edge 0 and edge N to all,
  // A4); the loop is kept rolled: one compact body for every edge (L0 instruction cache, see the header).
  template <int DEPTH>
  __device__ __forceinline__ void thick(int N, double& Sx, double& Sy, double& Ss) {
    SpinAcc<DEPTH> acc;
    {
      Quat q = pop();                               // edge 0 starts every level
      acc.Q[0] = q;
#pragma unroll
      for (int l = 1; l < DEPTH; ++l) { q = quat_double(q); acc.Q[l] = q; }
    }
#pragma unroll 1
    for (int i = 1; i <= N; ++i) {
      Quat q = pop();
      acc.Q[0] = quat_mul(q, acc.Q[0]);
      acc.template fold_dynamic<1>(i, q);
    }
    acc.finish(Sx, Sy, Ss);
  }
};

// registers: 14 warp pairs per SM (28 warps, 7 per sub-partition) need <= 72 registers per thread;
// depths 5 and 6 carry 40 / 48 registers of level products and get a looser bound.
template <int DEPTH> struct PairCfg {
  static constexpr int PAIRS = 1;                      // warp pairs per block (32 particles)
  static constexpr int THREADS = 64 * PAIRS;
  static constexpr int MIN_BLOCKS = DEPTH <= 4 ? 14 : (DEPTH == 5 ? 12 : 10);
};

// ---- the two roles ---------------------------------------------------------------------------
template <int SPLIT>
__device__ __forceinline__ void orbit_role(const TrackArgs& a, const DevElem* tab, const uint32_t* seq, double* ring_lane,
                                           uint8_t* flag_lane, long long j, bool valid) {
  Chan ch{ring_lane, 0};
  State z;
  z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
  z.Sx = z.Sy = z.Ss = 0.0;
  if (valid) {
    z.X = a.p[0][j]; z.Px = a.p[1][j]; z.Y = a.p[2][j]; z.Py = a.p[3][j]; z.T = a.p[4][j]; z.Pt = a.p[5][j];
  }
  Ref ref;
  ref_set(ref, a.E0, a.mass);
  ref.E0lo = a.E0lo;
  PCon pc;
  pcon_set(pc, z.Pt, ref, a.G);
  bool lost = false;
  PushSpin spin(ch);
  for (long long turn = 0; turn < a.n_turns; ++turn) {
#pragma unroll 1
    for (int ie = 0; ie < a.n_seq; ++ie) {
      const uint32_t cur = seq[ie];
      const DevElem& e = tab[cur >> 8];
      const bool ok = element_step<SPLIT, 2>((int)(cur & 0xffu), z, e, pc, ref, a.G, spin);
      if (!ok) {
        // A15: the particle is lost.  The warp must stay in step with its partner, so the lane goes on
        // with the reference orbit (all zeros); nothing of it is stored.
        lost = true;
        z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
        pcon_set(pc, 0.0, ref, a.G);
      }
    }
  }
  spin.flush();
  *flag_lane = lost ? 1 : 0;
  if (valid) {
    if (lost) {
      a.lost[j] = 1;
    } else {
      a.p[0][j] = z.X; a.p[1][j] = z.Px; a.p[2][j] = z.Y; a.p[3][j] = z.Py; a.p[4][j] = z.T; a.p[5][j] = z.Pt;
    }
  }
}

template <int DEPTH>
__device__ __forceinline__ void spin_role(const TrackArgs& a, const DevElem* tab, const uint32_t* seq, double* ring_lane,
                                          long long j, bool valid, double& Sx, double& Sy, double& Ss) {
  Chan ch{ring_lane, 0};
  if (valid) { Sx = a.p[6][j]; Sy = a.p[7][j]; Ss = a.p[8][j]; }
  PopSpin spin(ch);
  spin.start();
  for (long long turn = 0; turn < a.n_turns; ++turn) {
#pragma unroll 1
    for (int ie = 0; ie < a.n_seq; ++ie) {
      const uint32_t cur = seq[ie];
      const DevElem& e = tab[cur >> 8];
      const int type = (int)(cur & 0xffu);
      if (type == K_SBEND || type == K_QUAD || type == K_MULT) {
        spin.template thick<DEPTH>(e.N, Sx, Sy, Ss);
      } else if (type == K_RBEND) {               // frame rotation, fringe kick, body, fringe kick, frame rotation
        quat_rotate(Quat{e.rb_qw[0], 0.0, e.rb_qy[0], 0.0}, Sx, Sy, Ss);
        Quat q = spin.pop();
        quat_rotate(q, Sx, Sy, Ss);
        spin.template thick<DEPTH>(e.N, Sx, Sy, Ss);
        q = spin.pop();
        quat_rotate(q, Sx, Sy, Ss);
        quat_rotate(Quat{e.rb_qw[1], 0.0, e.rb_qy[1], 0.0}, Sx, Sy, Ss);
      } else if (type == K_SOLENOID) {            // entrance kick, body, exit kick
        Quat q = spin.pop();
        quat_rotate(q, Sx, Sy, Ss);
        spin.template thick<DEPTH>(e.N, Sx, Sy, Ss);
        q = spin.pop();
        quat_rotate(q, Sx, Sy, Ss);
      } else if (type == K_THIN || type == K_FRINGE) {
        Quat q = spin.pop();
        quat_rotate(q, Sx, Sy, Ss);
      } else if (type == K_SNAKE) {
        Quat q{e.qw, e.qx, e.qy, e.qs};
        quat_rotate(q, Sx, Sy, Ss);
      }
    }
  }
}

template <int SPLIT, int DEPTH>
__global__ void __launch_bounds__(PairCfg<DEPTH>::THREADS, PairCfg<DEPTH>::MIN_BLOCKS) track_pair_kernel(const TrackArgs a) {
  constexpr int PAIRS = PairCfg<DEPTH>::PAIRS;
  static_assert(PAIRS == 1, "barrier ids 0..3 serve one pair per block");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // layout: ring[PAIRS] | lost flags [PAIRS*32] | element table | sequence (when it fits)
  double* ring = reinterpret_cast<double*>(smem_raw);
  uint8_t* flag = smem_raw + PAIRS * PAIR_RING_BYTES;
  unsigned char* tab_raw = flag + PAIRS * 32;
  const DevElem* tab = a.tab;
  const uint32_t* seq = a.seq;
  {
    size_t off = 0;
    if (a.use_smem_tab) {
      const int nw = a.n_unique * (int)(sizeof(DevElem) / sizeof(double));
      const double* src = reinterpret_cast<const double*>(a.tab);
      double* dst = reinterpret_cast<double*>(tab_raw);
      for (int i = threadIdx.x; i < nw; i += blockDim.x) dst[i] = src[i];
      tab = reinterpret_cast<const DevElem*>(tab_raw);
      off = (size_t)a.n_unique * sizeof(DevElem);
    }
    if (a.use_smem_seq) {
      uint32_t* sseq = reinterpret_cast<uint32_t*>(tab_raw + off);
      for (int i = threadIdx.x; i < a.n_seq; i += blockDim.x) sseq[i] = a.seq[i];
      seq = sseq;
    }
    __syncthreads();
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // warp 0 = orbit, warp 1 = spin; swapped in every other group of four hardware warp slots, so that each
  // sub-partition (slot % 4) runs both roles and carries the same load (measured: 7 % faster than fixed roles)
  const int pair = 0;
  int swap;
  {
    int* sw = reinterpret_cast<int*>(flag);
    if (threadIdx.x == 0) {
      unsigned hw;
      asm volatile("mov.u32 %0, %%warpid;" : "=r"(hw));
      *sw = (int)((hw >> 2) & 1u);
    }
    __syncthreads();
    swap = *sw;
    __syncthreads();      // flag[] is reused for the lost flags at the end
  }
  const int is_spin = (warp ^ swap) & 1;
  double* ring_lane = ring + pair * (PAIR_SLOTS * PAIR_EDGE_DOUBLES) + lane;
  uint8_t* flag_lane = flag + pair * 32 + lane;
  const long long j = ((long long)blockIdx.x * PAIRS + pair) * 32 + lane;
  const bool valid = j < a.n && !a.lost[j];
  double Sx = 0.0, Sy = 1.0, Ss = 0.0;
  if (!is_spin) {
    orbit_role<SPLIT>(a, tab, seq, ring_lane, flag_lane, j, valid);
  } else {
    spin_role<DEPTH>(a, tab, seq, ring_lane, j, valid, Sx, Sy, Ss);
  }
  __syncthreads();      // the orbit threads' lost flags are visible
  if (is_spin && valid && !*flag_lane) { a.p[6][j] = Sx; a.p[7][j] = Sy; a.p[8][j] = Ss; }
}

}  // namespace gst
